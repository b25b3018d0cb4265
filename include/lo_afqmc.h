/* lo_afqmc.h -- C ABI of the B200-native LO-AFQMC local-energy library (liblo_afqmc.so).
 *
 * The library evaluates, for a batch of walkers, the phaseless-AFQMC local energy with a
 * single-determinant trial (arxiv 2202.00832; citations are /root/reference/PAPER.md lines):
 *
 *   Theta_w = Phi_w (Psi^T Phi_w)^-1                                  Eq. 15
 *   E1      = c1 sum_{i,p} hbar_ip Theta_pi                           Eq. 8 one-body part
 *   X^g     = sum_{i,p} Lbar^g_ip Theta_pi ;  E_J = cJ sum_g (X^g)^2  Eq. 16 Coulomb part
 *   E_K     = -cK sum_{i<=j} m_ij sum_{K<=r_ij} sigma_K (U^{ij T} Theta_j)_K (W^{ij} Theta_i)_K
 *                                                                     Eq. 18, 19/22 exchange part
 *   E_L     = E1 + E_J + E_K
 *
 * with Lbar^g_ip = sum_q L^g_pq Psi_qi, Y^{ij}_pq = sum_g Lbar^g_ip Lbar^g_jq
 * = U sigma W truncated to the r_ij singular values > threshold (Eq. 18), m_ij = 1 (i=j) or 2 (i<j).
 * Closed shell (n_spin=1): c1=2, cJ=2, cK=1.  Unrestricted (n_spin=2): c1=1, cJ=1/2 with X summed over both
 * spins, cK=1/2 with same-spin pairs only (Eq. 10 with explicit spin sums).  Readings of the paper's silent
 * points are listed in DESIGN.md.
 *
 * Conventions: all matrices row-major (C order); complex128 = two doubles (re, im) interleaved.
 * "host" / "device" is stated for every pointer.  No call throws; every call returns a lo_status and
 * lo_last_error() gives a thread-local message for the last failure.  The library never frees or keeps
 * caller memory.  There is no CPU fallback: lo_local_energy* need a factor set built with device >= 0.
 * A lo_factors handle owns ONE workspace (Theta panels, partial sums): calls on the same handle must be serialised by
 * the caller (stream order on one stream is enough); different handles, e.g. lo_retruncate copies, are independent.
 * lo_local_energy / lo_local_energy_cas / lo_propagator only enqueue work on the given stream, so a step can be captured
 * in a CUDA graph (with timing disabled).
 */
#ifndef LO_AFQMC_H
#define LO_AFQMC_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lo_factors lo_factors; /* opaque; owns every host and device allocation it makes */

typedef enum {
    LO_OK = 0,
    LO_EINVAL = 1,    /* bad shape / NULL / misaligned pointer / n_w > max_walkers: nothing was launched */
    LO_ENOMEM = 2,    /* host or device allocation failed */
    LO_ECUDA = 3,     /* a CUDA call failed, or the factor set has no device (built with device < 0) */
    LO_EINTERNAL = 5  /* the setup SVD did not converge (see lo_last_error) */
} lo_status;

typedef struct {
    int N, n_chol, n_spin, n_occ[2];
    int N_pad;                       /* N rounded up to the K tile (16) */
    long long n_pairs[2];            /* pairs i<=j per spin */
    long long sum_rank[2];           /* sum of r_ij per spin (R of SURVEY 8d) */
    long long sum_rank_padded;       /* rows of the packed factor arrays (ranks padded to x8) */
    int max_rank, min_rank;
    unsigned long long factor_bytes; /* device bytes of packed U, W, weights and the tile table */
    unsigned long long lbar_bytes;   /* device bytes of the half-rotated Cholesky operand [Lbar; hbar] */
    unsigned long long workspace_bytes;
    double threshold;
    int device, max_walkers;
    int setup_on_gpu;                /* 1 when pair Gram + SVD ran on the device */
    long long n_tiles;               /* row tiles of the exchange grouped GEMM */
    int svd_sweeps_max;              /* pair-block SVD: most sweeps any block took (incl. the final checking sweep) */
    double svd_offdiag_max;          /* and the largest normalised off-diagonal |g_p.g_q|/(|g_p||g_q|) left at the end */
    double setup_seconds;            /* wall time of lo_setup, and of its pair Gram + SVD part */
    double setup_svd_seconds;
    int rsvd_sketch;                 /* sketch rows of LO_SETUP_RANDOMIZED_SVD (0: full SVDs only) */
    long long n_pairs_rsvd;          /* pair blocks whose randomised sketch was accepted */
    long long n_pairs_prescreened;   /* pairs given rank 0 by the rigorous pre-SVD norm bounds (no SVD was run for them) */
    long long n_pairs_energy_screened; /* pairs dropped by lo_screen_pairs (m_ij sigma_1 <= energy_screen_cutoff) */
    double energy_screen_cutoff;     /* 0 when no energy screen was applied */
    double energy_screen_bound;      /* cK sum over the dropped pairs of m_ij sigma_1: |dE_K| <= this x max_i |Theta_i|^2 */
    int exchange_mode;               /* LO_EXCHANGE_DMMA / LO_EXCHANGE_INT8 (lo_set_exchange_mode) */
    unsigned long long int8_bytes;   /* device memory of the INT8 digit slices (0 until LO_EXCHANGE_INT8 was first set) */
} lo_info;

/* Kernel indices for lo_timing_get */
enum { LO_K_OVERLAP = 0, LO_K_INVERSE = 1, LO_K_THETA = 2, LO_K_COULOMB = 3, LO_K_EXCHANGE = 4, LO_K_FINAL = 5, LO_K_PROPAGATOR = 6, LO_K_COUNT = 7 };

/* S0 setup (untimed, deterministic): half-rotation, per-pair Y^{ij}, SVD,
 * truncation sigma_K > threshold (strict, absolute; Eq. 18), sorting pairs by rank, padding
 * ranks to multiples of 8, packing and upload.
 *   h      host [N][N] symmetric.         L      host [n_chol][N][N], every slice symmetric.
 *   psi_a  host [N][n_occ[0]], orthonormal columns (real trial).   psi_b  host [N][n_occ[1]] or NULL if n_spin==1.
 *   threshold >= 0 (T_SVD, same units as the integrals).
 *   device >= 0: CUDA device that will hold the factor set and workspace for up to max_walkers walkers.
 *   device <  0: host-only factor set (accessors work; lo_local_energy* return LO_ECUDA).
 *   flags  bit 0 (LO_SETUP_GPU_SVD): run the pair Gram matrices and their SVDs (block one-sided Jacobi, DMMA) on the device
 *          (needs device >= 0); otherwise they run on the host with OpenMP.
 * On success *out owns everything; release with lo_free. */
#define LO_SETUP_GPU_SVD 1
/* flags bit 1 (LO_SETUP_PROPAGATOR, needs device >= 0): also keep the Cholesky vectors L on the device, packed for
 * lo_propagator (upper triangle p<=q, K-major: [N(N+1)/2][n_chol]), and reserve its output buffer. */
#define LO_SETUP_PROPAGATOR 2
/* flags bit 2 (LO_SETUP_NO_PRESCREEN): switch the rigorous pre-SVD pair screen off.  By default a pair (i,j) with
 *     sigma_1(Y^{ij}) <= |Y^{ij}|_F <= sum_g |Lbar^g_i|_2 |Lbar^g_j|_2 <= threshold
 * ("screening pairs of electrons") is given rank 0 without forming its block (second bound) or without
 * running its SVD (first bound); the factor rows, weights, ranks and tiles are the same with and without the screen
 * (Eq. 18 would discard every singular value of such a pair); only the recorded first discarded singular value of a
 * screened pair is its bound instead of sigma_1.  lo_info.n_pairs_prescreened counts them. */
#define LO_SETUP_NO_PRESCREEN 4
/* flags bit 3 (LO_SETUP_RANDOMIZED_SVD, "approximate versions of the singular value decomposition,
 * which would reduce the scaling of this step significantly"): every pair block is first decomposed through
 * a randomised sketch of k rows (Gaussian test matrix from a fixed counter-based generator; range finder, projected
 * block, small SVD; k = 16 x (bits 8..15 of flags), default 64, at most 128 and N/4) whose a-posteriori error
 * |Y - U^T sigma W|_F is formed explicitly; a block is accepted only when that error is <= 16 N 2^-53 |Y|_F, i.e. when its
 * numerical rank is below k and the sketch IS its SVD to working accuracy (every singular value of Y is within the error of
 * a returned one).  All other blocks are decomposed by the full method.  The factor set is therefore the same to rounding
 * (tests pin it to LAPACK either way); what changes is the setup time of low-rank problems.  lo_info.n_pairs_rsvd counts
 * the accepted blocks. */
#define LO_SETUP_RANDOMIZED_SVD 8
lo_status lo_setup(int N, int n_chol, int n_spin, const int n_occ[2], const double* h, const double* L,
                   const double* psi_a, const double* psi_b, double threshold, int device, int max_walkers,
                   unsigned flags, lo_factors** out);

lo_status lo_info_get(const lo_factors* f, lo_info* info);

/* r[k] = r_ij for the pairs of one spin in row-major i<=j order ((0,0),(0,1),...,(0,O-1),(1,1),...); host [n_pairs]. */
lo_status lo_ranks(const lo_factors* f, int spin, int* r);

/* Host copy of the factors of pair (i<=j) of one spin, so that a checker can evaluate on THIS factor set:
 * U host [r][N] (row K = left singular vector over p), sigma host [r] (descending), W host [r][N]. Any may be NULL. */
lo_status lo_factor_pair(const lo_factors* f, int spin, int i, int j, double* U, double* sigma, double* W);

/* All factors of one spin in lo_ranks order, rows back to back: U,W host [sum_rank][N], sigma host [sum_rank]. */
lo_status lo_factor_all(const lo_factors* f, int spin, double* U, double* sigma, double* W);

/* New factor set with a looser threshold (>= the one f was built with): prefix truncation of every pair,
 * re-sorted and re-packed; Lbar/hbar are shared by reference counting.  Used for threshold sweeps. */
lo_status lo_retruncate(const lo_factors* f, double looser_threshold, lo_factors** out);

/* Energy screen of pairs ("screening pairs of electrons, and only including those
 * that contribute meaningfully to the total energy"): new factor set, same threshold, in which every pair with
 *     m_ij sigma_1^{ij} <= pair_cutoff        (m_ij = 2 - delta_ij, sigma_1 = largest kept singular value)
 * has rank 0.  An approximation with an explicit knob (pair_cutoff = 0 changes nothing): since
 * |sum_K sigma_K a_K b_K| <= sigma_1 |Theta_i|_2 |Theta_j|_2, a walker's E_K moves by at most
 * cK sum_dropped m_ij sigma_1 |Theta_i|_2 |Theta_j|_2 <= lo_info.energy_screen_bound x max_i |Theta_i|_2^2.
 * lo_info.n_pairs_energy_screened counts the dropped pairs.  Lbar/hbar are shared with f. */
lo_status lo_screen_pairs(const lo_factors* f, double pair_cutoff, lo_factors** out);

/* S1-S5: local energies of n_w walkers.  Asynchronous on `stream`; allocates nothing; no host sync.
 *   phi_a  device complex128 [n_w][N][n_occ[0]] (walker-major; columns = orbitals), 16-byte aligned.
 *   phi_b  device complex128 [n_w][N][n_occ[1]] or NULL when n_spin==1.
 *   E_L, E1, E_J, E_K  device complex128 [n_w]; E_L required, parts may be NULL.
 *   walker_status  device int32 [n_w] or NULL; nonzero = singular overlap Psi^T Phi, that walker's energies are NaN.
 *   stream  cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream. */
lo_status lo_local_energy(const lo_factors* f, int n_w, const void* phi_a, const void* phi_b, void* E_L, void* E1,
                          void* E_J, void* E_K, int* walker_status, void* stream);

/* Same computation with HOST buffers: copies phi to the device, runs lo_local_energy, copies
 * E[n_w][4] = {E_L, E1, E_J, E_K} (complex128) and status back, and synchronises.  Pinned host memory makes the
 * copies asynchronous with respect to each other; pageable memory works too.
 * The batch runs in up to 4 walker chunks: the host-to-device copies go on a private stream that first waits for
 * everything already queued on `stream`, the kernels of chunk c run on `stream` under the copy of chunk c+1.  Both streams
 * are synchronised before the call returns, also when it fails.  Calls on one handle must be serialised by the caller
 * (one workspace).  After this call lo_coulomb_x holds the X of the LAST chunk only (columns 0.. of that chunk). */
lo_status lo_local_energy_host(const lo_factors* f, int n_w, const void* phi_a_host, const void* phi_b_host,
                               void* E_host, int* status_host, void* stream);

/* X^g_w = sum_{ip} Lbar^g_ip Theta_pi of the last lo_local_energy call (the force-bias contraction of
 * PAPER.md:34): device complex128 [n_chol][ld] with ld returned in *ld (walker index fastest).
 * Valid until the next call on this factor set. */
lo_status lo_coulomb_x(const lo_factors* f, const void** X_dev, int* ld);

/* SURVEY 8(f) NEXT-3, the paper-literal energy expression: with LO_COULOMB_COMPRESSED the Coulomb term of every later
 * lo_local_energy* call is evaluated from the SVD-compressed pair factors as well,
 *   E_J^LO = 2 sum_{i<=j} m_ij sum_{K<=r_ij} sigma_K (U^{ij T} Theta_i)_K (W^{ij} Theta_j)_K     (closed shell)
 * (Eq. 19/22 first term "4 Q_{K,L,i} Q_{K,R,j}"; the four projections per pair of PAPER.md:181
 * come from the same staged tiles as the exchange), so E_J carries the truncation error too.  The default
 * LO_COULOMB_CHOLESKY evaluates E_J = cJ sum_g (X^g)^2 exactly (Eq. 16).  X^g (lo_coulomb_x) and E1 are formed in both
 * modes.  Closed shell only: an unrestricted factor set holds same-spin pairs only (LO_EINVAL). */
#define LO_COULOMB_CHOLESKY 0
#define LO_COULOMB_COMPRESSED 1
lo_status lo_set_coulomb_mode(lo_factors* f, int mode);

/* Arithmetic of the two heavy contractions of every later lo_local_energy* call on this (device-resident) factor set.
 *   LO_EXCHANGE_DMMA (default): the exchange projections a = U Theta_j, b = W Theta_i (Eq. 18) and the Coulomb / one-body
 *     contraction X^g = sum L^g_op Theta_po (Eq. 16) as FP64 tensor-pipe GEMMs (mma.sync m8n8k4.f64), as written.
 *   LO_EXCHANGE_INT8: the same contractions from exact INT8 digit slices on the tcgen05 tensor cores (Ozaki-type splitting:
 *     every row of U, W, Lbar (per orbital) and Theta^T is scaled by a power of two and cut into 7 signed 7-bit digits; the 28
 *     digit products with digit-index sum <= 6 are exact int32 GEMMs accumulated in TMEM; recombination, sigma weights, the a.b
 *     reduction and E_J = sum_g (X^g)^2 in fp64).  Not bit-identical to the DMMA route: the projections carry an absolute error
 *     of about 2^-47 |row|_max |Theta row|_max N, the energies agree to 1e-12 .. 1e-11 of |E_L| on the BASELINE configs (DESIGN.md
 *     section 6b; the parity tests hold this route to the same 1e-10 as the default).  The first call slices the factor rows and
 *     Lbar once (extra device memory: 7/8 of the factor and Lbar bytes + 7 bytes per Theta^T element, lo_info.int8_bytes) and
 *     is synchronous; LO_ENOMEM leaves the set in LO_EXCHANGE_DMMA mode.  Combines with LO_COULOMB_COMPRESSED (four projections
 *     per pair from the same digits).  Ignored by lo_local_energy_cas, which keeps its DMMA kernels.  lo_propagator follows the mode as well (factor sets built with
 *     LO_SETUP_PROPAGATOR: the GEMM B = Lt x from digits of Lt, + 7/8 of its bytes, and of the fields).
 * Host-only factor sets: LO_EINVAL. */
#define LO_EXCHANGE_DMMA 0
#define LO_EXCHANGE_INT8 1
lo_status lo_set_exchange_mode(lo_factors* f, int mode);

/* SURVEY 8(f) NEXT-2, multi-determinant (CAS-type) trial |Psi_T> = sum_d c_d |d> of closed-shell determinants (the
 * same excitation string in both spins), each at most max_exc (<= 8) excitations from the reference:
 *   E = sum_d w_d E^d / sum_d w_d,  w_d = c_d <d|Phi>   (Eq. 12 with Eq. 13, applied to every energy term)
 * evaluated by direct summation over determinants ("direct summation"); the determinants' overlaps and
 * half-rotated Green's functions come from Sherman-Morrison-Woodbury updates of the reference (Eq. 20),
 * and every (walker, determinant) runs through the Coulomb / exchange kernels as one virtual walker.  The factor set
 * must have been built (n_spin = 1) with psi = [reference occupied orbitals | active virtual orbitals], i.e.
 * n_occ[0] = n_ref + n_virt orthonormal columns, and max_walkers >= max_real_walkers * n_det.
 *   holes  host int32 [n_det][max_exc]: replaced column positions of the reference (< n_ref), -1 padding at the end
 *   parts  host int32 [n_det][max_exc]: the orbital (column of psi, in [n_ref, n_occ[0])) put in that position
 *   coef   host [n_det]: c_d.   Determinant 0 is normally the reference (no excitation).
 * lo_set_cas_trial copies the lists and reserves the workspace; it may be called again to replace the trial.
 * lo_local_energy_cas: phi device complex128 [n_w][N][n_ref]; E_L (required), E1, E_J, E_K, ovlp device complex128
 * [n_w] (ovlp = sum_d w_d / <reference|Phi>, the trial overlap in units of the reference overlap); walker_status as in
 * lo_local_energy.  A determinant with a singular overlap contributes nothing.  Asynchronous; allocates nothing.
 * Closed-shell factor sets (n_spin = 1) use the same string for both spins (w_d = c_d det^2).
 * mode LO_CAS_DIRECT: cost = n_det x the single-determinant evaluation; needs max_walkers >= max_real_walkers * n_det.
 * mode LO_CAS_SMW_ENERGY: the rearranged sums of Eq. 21-23: every Theta^d column is the reference
 *   column plus a combination of the active (hole) columns of Theta0 = Phi A^-1, so for each pair (x<=y) the projections
 *   of U^{xy}, W^{xy} onto the panel set {x, y} u active ("Q_L^int") are formed ONCE per walker, contracted
 *   over the singular index into S^{xy}[c][c'] = sum_K sigma_K (U_K.Theta0_c)(W_K.Theta0_c'), and each determinant's
 *   exchange AND Coulomb pair energies (Eq. 22: both terms from the compressed factors, as LO_COULOMB_COMPRESSED) are
 *   small bilinear forms in S; E1 likewise from hbar.Theta0 intermediates.  Leading cost (2 + n_active)/2 x the
 *   4-projection single-determinant evaluation, independent of n_det.  Up to 6 distinct hole columns (active occupied
 *   orbitals) take one pass; 7..12 are cut into groups of 3 and take one pass per pair of groups (6 passes for 9, 10 for 12). */
#define LO_CAS_DIRECT 0
#define LO_CAS_SMW_ENERGY 1
lo_status lo_set_cas_trial(lo_factors* f, int n_ref, int n_det, int max_exc, const int* holes, const int* parts,
                           const double* coef, int max_real_walkers, int mode);
/* Unrestricted trial (factor set with n_spin = 2, either mode): determinant d = |alpha string d> |beta string d>.
 * lo_set_cas_trial gives the alpha strings (reference = the first n_ref columns of psi_a), lo_set_cas_trial_beta the
 * beta strings of the same n_det / max_exc (reference = the first n_ref_b columns of psi_b); w_d = c_d det_a det_b.
 * LO_CAS_DIRECT: every (walker, determinant) is one virtual walker of the unrestricted path (Eq. 10 with explicit spin
 * sums).  LO_CAS_SMW_ENERGY (the paper's own use: open-shell systems with 200-determinant trials): the
 * exchange of each spin from that spin's S intermediates as above; the Coulomb term by the Cholesky route (an
 * unrestricted factor set holds no opposite-spin pair blocks): X^{g,d}_s = X0^g_s + sum_k sum_x (G_d[k][x] - [x = hole k])
 * Z_s[hole k][g][x] with Z_s[a][g][x] = Lbar^g_x . Theta0_{s,a} formed once per walker by one GEMM per spin, and
 * E_J^d = 1/2 sum_g (X^{g,d}_alpha + X^{g,d}_beta)^2; at most 6 distinct hole columns per spin; the Z workspace takes
 * 8 (n_active padded to 2/4/6) x 2 max_real_walkers(rounded up to 64) x (n_chol padded) x (n_occ[0]+n_occ[1]) bytes per spin. */
lo_status lo_set_cas_trial_beta(lo_factors* f, int n_ref_b, const int* holes_b, const int* parts_b);
/* phi_b: device complex128 [n_w][N][n_ref_b] for an unrestricted trial, NULL otherwise. */
lo_status lo_local_energy_cas(const lo_factors* f, int n_w, const void* phi, const void* phi_b, void* E_L, void* E1,
                              void* E_J, void* E_K, void* ovlp, int* walker_status, void* stream);

/* SURVEY 8(f) NEXT-1, propagator formation: B_w = sum_g x^g_w L^g ("forming the propagation matrix
 * (B = sum_alpha x_alpha L_alpha), scaling as X M^2"), for n_w walkers at once as one real x
 * complex FP64 GEMM on the DMMA pipe ([N(N+1)/2 x n_chol] x [n_chol x 2 n_w]).  Every L^g is symmetric, so B_w is
 * (complex) symmetric and only the upper triangle is formed.
 *   x_dev  device complex128 [n_w][n_chol] (walker-major): the shifted auxiliary fields of each walker.
 * The result stays in a library-owned device buffer (lo_propagator_buffer): complex128 [n_rows][ld], row
 * r(p,q) = p*N - p*(p-1)/2 + (q-p) for p<=q, walker index fastest; valid until the next lo_propagator call.
 * Needs a factor set built with LO_SETUP_PROPAGATOR (else LO_EINVAL).  Asynchronous on `stream`; allocates nothing. */
lo_status lo_propagator(const lo_factors* f, int n_w, const void* x_dev, void* stream);
lo_status lo_propagator_buffer(const lo_factors* f, const void** B_dev, int* ld, long long* n_rows);
/* B_w of the last lo_propagator call for one walker, unpacked to the full symmetric matrix, for tests:
 * host complex128 [N][N].  Synchronises the device. */
lo_status lo_propagator_host(const lo_factors* f, int w, void* B_host);

/* Theta of the last call, for tests: host complex128 [n_w][N][n_occ[spin]] (walker-major, same layout as phi). */
lo_status lo_theta_host(const lo_factors* f, int spin, int n_w, void* theta_host);

/* Per-kernel device timing: when enabled, every lo_local_energy call brackets each of its kernels with CUDA
 * events on `stream`; lo_timing_get synchronises those events and returns the accumulated milliseconds and launch
 * counts per kernel (LO_K_*), then resets them. */
lo_status lo_timing_enable(lo_factors* f, int enable);
lo_status lo_timing_get(lo_factors* f, double ms[LO_K_COUNT], long long launches[LO_K_COUNT]);

/* Algorithmic FP64 flops of ONE walker's local energy on this factor set: per step S1..S4. */
lo_status lo_flops_per_walker(const lo_factors* f, double flops[LO_K_COUNT]);

/* In-run roofline denominators (microbenchmarks on `device`):
 *   kind 0: FP64 tensor pipe, register-resident DMMA.8x8x4 loop  -> *value in TFLOP/s
 *   kind 1: FP64 FMA pipe, register-resident DFMA loop           -> *value in TFLOP/s
 *   kind 2: HBM stream copy (read+write bytes)                   -> *value in GB/s
 * and one gated experiment that is NOT part of any product path: an FP64-accurate 128 x 128 x 384 GEMM
 * tile from 6 x 6 signed 7-bit INT8 slices on the 5th-generation tensor cores (tcgen05.mma kind::i8, TMEM accumulators, fp64
 * recombination), operands resident in shared memory:
 *   kind 3: microseconds per tile                                -> *value in us
 *   kind 4: max |C - C_fp64| / max |C_fp64| of that tile         -> *value dimensionless */
lo_status lo_measure_peak(int device, int kind, double* value);

/* Allocation-free S1 for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): Theta = Phi (Psi^T Phi)^-1 (Eq. 15) for a batch of walkers with NO factor set and NO
 * allocation of any kind -- the same kernels as step S1 of lo_local_energy (k_overlap, k_inverse, k_theta); their
 * scratch, the overlap matrices A_w = Psi^T Phi_w inverted in place (16 n_w n_occ^2 bytes), lives in a file-scope
 * `static __device__` array of LO_NOALLOC_SCRATCH_BYTES (4 MiB) that every GPU holds from the moment it loads the library
 * until the process exits.
 *   device            CUDA device the pointers belong to
 *   N, n_occ, n_w     basis functions, occupied orbitals (1 <= n_occ <= N), walkers (>= 1);
 *                     16 n_w n_occ^2 > LO_NOALLOC_SCRATCH_BYTES is refused with LO_EINVAL (split the batch)
 *   psi_dev           device fp64 [N][n_occ] row-major (trial orbitals, real)
 *   phi_dev           device complex128 [n_w][N][n_occ] (walker-major, as lo_local_energy)
 *   thetaT_dev        OUT, device fp64 [n_occ][ld_w][N_pad], N_pad = N rounded up to a multiple of 16: the Theta^T panel layout
 *                     of the library, thetaT[(i ld_w + 2 w + c) N_pad + p] = (c ? Im : Re) Theta_w[p][i]; entries
 *                     p in [N, N_pad) are written as zeros, rows 2 w + c >= 2 n_w are not touched.  ld_w >= 2 n_w, even.
 *   status_dev        OUT, device int [n_w]: 1 for a walker whose overlap matrix is singular (its Theta is NaN), else 0
 *   stream            cudaStream_t; the call is asynchronous on it
 * lo_theta_noalloc_init(device) fetches the device address of the scratch array (cudaGetSymbolAddress) and sets the kernels'
 * shared-memory attributes; call it once per device BEFORE any stream capture (lo_theta_noalloc calls it itself on first use
 * otherwise).  Neither function calls cudaMalloc, cudaFree or an allocating library routine.
 * The scratch array is shared by every call on a device and keeps the last call's contents; nothing in it has to start at
 * zero (every entry a call reads it has written first), but two calls that overlap on the GPU (different streams, or
 * concurrent graph launches) race on it: serialise them.
 * Errors: LO_EINVAL (arguments, size beyond the maximum), LO_ECUDA. */
#define LO_NOALLOC_SCRATCH_BYTES (4u << 20)
lo_status lo_theta_noalloc_init(int device);
lo_status lo_theta_noalloc(int device, int N, int n_occ, int n_w, const double* psi_dev, const void* phi_dev, double* thetaT_dev, int ld_w,
                           int* status_dev, void* stream);

void lo_free(lo_factors* f);
const char* lo_last_error(void);
const char* lo_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LO_AFQMC_H */
