// lo_exchange_i8.cu -- the exchange term (Eq. 18 / 19 / 22 exchange part) on the 5th-generation tensor
// cores: fp64-accurate projections a = U Theta_j, b = W Theta_i from INT8 digit slices (tcgen05.mma kind::i8, int32
// accumulators in TMEM), the sigma-weighted complex a.b reduction fused into the TMEM read-out.  Opt-in
// (lo_set_exchange_mode(f, LO_EXCHANGE_INT8)); the default exchange stays the FP64 DMMA kernel k_exchange.
//
// Scheme (Ozaki-type splitting).  A row x of an operand is scaled by a power of two, |x| 2^-e < 1,
// and cut into XI_S = 7 signed digits of 7 bits,  x = 2^e sum_s d_s 2^-(7 s + 6),  |d_s| <= 64  (exact: the remainder after
// 7 digits is below 2^(e-49)).  Digit matrices are int8, their products are exact in int32 (|sum| <= 7 * N * 2^12), and
//     a_K[m] = 2^(e_m + e_K) sum_{g <= 6} 2^-(7 g + 12) D_g[m][K],   D_g = sum_{s + t = g} dTheta_s dU_t^T
// keeps the 28 digit products with s + t <= 6 in 7 accumulators ("groups").  Rows of Theta^T (walker w, re / im) share one
// exponent per (orbital, walker), so the complex product a_K b_K carries one power of two per walker.
//
// Mapping.  M side (TMEM lanes) = 128 walker rows (64 walkers x re/im) of a Theta^T panel, N side (TMEM columns) = the <= 64
// factor rows of one exchange tile, K = basis index in blocks of 32.  A work item (tile, walker block) runs two phases,
// a then b, each streaming K once with all 7 groups live in TMEM (7 x 64 = 448 of the 512 columns).  One CTA per SM,
// 12 warps: warp 0 (one lane) feeds a 5-stage ring with cp.async.bulk copies of pre-tiled slices (Theta: 7 x 4 KB, factor
// rows: 7 x 2 KB per stage), warp 1 (one lane) issues the MMAs and commits stages / accumulators to mbarriers, warps 4..11
// read TMEM (lane quadrant = warp % 4, column half = (warp - 4) / 4), merge the 7 groups of a column exactly in 64-bit integers, convert
// the two partial sums to fp64 (the FP64 pipe, 64 FMA / clock / SM, bounds the read-out) and, in phase b, multiply straight
// into the weighted dot with the a values they hold in registers (own row and the re/im partner row), so b is never stored.
// Per-CTA partial sums are updated in a fixed order by their owning thread: results are bitwise repeatable.
//
// Operand slices in HBM, in the shared-memory layout of a K-major, unswizzled tcgen05 operand (core matrix = 8 rows x 16 bytes):
//   Thq [(o * NBcap + nb)][kb][s][(r/8)*256 + (k/16)*128 + (r%8)*16 + k%16]   r = 2 (w % 64) + c < 128, k < 32   (per call)
//   Uq, Wq [tile][kb][s][same with r < 64]                                      rows of the tile, zero beyond them   (setup)
//   thScale [o][w] = 2^e of the Theta rows,  wq [row] = wgt[row] 2^(eU + eW)   (wgt = -cK m_ij sigma_K, lo_internal.h)
#include <algorithm>
#include <cstdlib>

#include "lo_device.cuh"

namespace lo {
namespace {

constexpr int XI_S = 7;                          // digits per operand
constexpr int XI_TH_BLK = 128 * 32;              // bytes of one (digit, K block) of a Theta walker block
constexpr int XI_F_BLK = 64 * 32;                // ... of the factor rows of a tile
constexpr int XI_TH_STAGE = XI_S * XI_TH_BLK, XI_F_STAGE = XI_S * XI_F_BLK;
constexpr int XI_STAGE = XI_TH_STAGE + XI_F_STAGE;          // 43008 bytes
constexpr int XI_STAGES = 5;
constexpr int XI_SMEM = XI_STAGES * XI_STAGE + 1024;
constexpr int XI_CAT = 4;                        // factor digits covered by one MMA (N <= 256)
constexpr int XI_TMEM_COLS = 512;                // 7 groups x 64 columns = 448, allocation sizes are powers of two

// ---- slicing ---------------------------------------------------------------------------------------------------------
// 16 consecutive k of one row -> one 16-byte chunk per digit
__device__ __forceinline__ void slice16(const double* __restrict__ src, double inv, int4 (&out)[XI_S]) {
    double res[16];
#pragma unroll
    for (int i = 0; i < 16; i += 2) {
        const double2 v = *reinterpret_cast<const double2*>(src + i);
        res[i] = v.x * inv;
        res[i + 1] = v.y * inv;
    }
#pragma unroll
    for (int s = 0; s < XI_S; ++s) {
        const double up = exp2(7.0 * s + 6.0), dn = exp2(-(7.0 * s + 6.0));
        int w[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            unsigned pk = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const double d = rint(res[4 * q + b] * up);
                res[4 * q + b] = fma(-d, dn, res[4 * q + b]);          // exact
                pk |= ((unsigned)(int)d & 0xFFu) << (8 * b);
            }
            w[q] = (int)pk;
        }
        out[s] = make_int4(w[0], w[1], w[2], w[3]);
    }
}

__device__ __forceinline__ int row_exponent(double mx) {
    // |x| 2^-e < 1 for every |x| <= mx, so that the leading digit rint(x 2^-e 2^6) lies in [-64, 64] like the others (one bit more
    // than |x| 2^-e <= 1/2 would keep);  rows of zeros and rows holding Inf / NaN (singular walkers, set to NaN by k_finalize) get e = 0
    return (mx > 0.0 && mx < 1e300) ? ilogb(mx) + 1 : 0;
}

// Theta^T panels -> Thq, thScale.  One warp per (orbital, walker): both rows (re, im) share the exponent.
__global__ void __launch_bounds__(256) k_slice_theta(const double* __restrict__ thT, int8_t* __restrict__ Thq, double* __restrict__ thScale,
                                                     int O_tot, int ldw, int N_pad, int KB, int NBcap, int Wcap, int n_wpad) {
    const int lane = threadIdx.x & 31;
    const long long gw = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int o = (int)(gw / n_wpad), w = (int)(gw % n_wpad);
    if (o >= O_tot) return;
    const double* r0 = thT + ((size_t)o * ldw + 2 * w) * N_pad;
    double mx = 0.0;
    bool bad = false;
    for (int i = lane; i < 2 * N_pad; i += 32) {
        const double a = fabs(r0[i]);
        bad |= !(a < 1e300);
        mx = fmax(mx, a);
    }
#pragma unroll
    for (int d = 16; d; d >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    bad = __any_sync(0xffffffffu, bad);
    const int e = bad ? 0 : row_exponent(mx);
    const double inv = bad ? 0.0 : scalbn(1.0, -e);
    if (lane == 0) thScale[(size_t)o * Wcap + w] = scalbn(1.0, e);
    const int nch = 2 * KB;                                   // 16-wide chunks per row
    int8_t* blk = Thq + (size_t)(o * NBcap + w / 64) * KB * XI_TH_STAGE;
    for (int task = lane; task < 2 * nch; task += 32) {
        const int c = task / nch, ch = task % nch, k0 = ch * 16, r = 2 * (w % 64) + c;
        int4 out[XI_S];
        if (k0 < N_pad && !bad) slice16(r0 + (size_t)c * N_pad + k0, inv, out);
        else {
#pragma unroll
            for (int s = 0; s < XI_S; ++s) out[s] = make_int4(0, 0, 0, 0);
        }
        int8_t* dst = blk + (size_t)(ch >> 1) * XI_TH_STAGE + (r >> 3) * 256 + (ch & 1) * 128 + (r & 7) * 16;
#pragma unroll
        for (int s = 0; s < XI_S; ++s) *reinterpret_cast<int4*>(dst + s * XI_TH_BLK) = out[s];
    }
}

// Factor rows -> Uq / Wq and their exponents.  grid = tiles, 8 warps; warp v handles rows v, v + 8, ... of the tile.
__global__ void __launch_bounds__(256) k_slice_factors(const double* __restrict__ F, const ExTile* __restrict__ tiles, int8_t* __restrict__ Fq,
                                                       int* __restrict__ eF, int N_pad, int KB) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const ExTile tile = tiles[blockIdx.x];
    const int nch = 2 * KB;
    int8_t* blk = Fq + (size_t)blockIdx.x * KB * XI_F_STAGE;
    for (int r = warp; r < 64; r += 8) {
        const bool live = r < tile.nfrag * 8;
        const double* src = F + (size_t)(tile.row0 + (live ? r : 0)) * N_pad;
        double mx = 0.0;
        if (live)
            for (int i = lane; i < N_pad; i += 32) mx = fmax(mx, fabs(src[i]));
#pragma unroll
        for (int d = 16; d; d >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        const int e = row_exponent(mx);
        const double inv = scalbn(1.0, -e);
        if (live && lane == 0) eF[tile.row0 + r] = e;
        for (int ch = lane; ch < nch; ch += 32) {
            const int k0 = ch * 16;
            int4 out[XI_S];
            if (live && k0 < N_pad) slice16(src + k0, inv, out);
            else {
#pragma unroll
                for (int s = 0; s < XI_S; ++s) out[s] = make_int4(0, 0, 0, 0);
            }
            int8_t* dst = blk + (size_t)(ch >> 1) * XI_F_STAGE + (r >> 3) * 256 + (ch & 1) * 128 + (r & 7) * 16;
#pragma unroll
            for (int s = 0; s < XI_S; ++s) *reinterpret_cast<int4*>(dst + s * XI_F_BLK) = out[s];
        }
    }
}

__global__ void k_i8_weights(const double* __restrict__ wgt, const int* __restrict__ eU, const int* __restrict__ eW, double* __restrict__ wq,
                             long long rows) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r < rows) wq[r] = scalbn(wgt[r], eU[r] + eW[r]);
}

// ---- the exchange kernel ---------------------------------------------------------------------------------------------
// shared-memory matrix descriptor, K-major, no swizzle: rows 16 bytes apart inside a core matrix, LBO = distance of the two
// 16-byte K halves, SBO = distance of consecutive 8-row groups; descriptor version 1 (sm_100)
__device__ __forceinline__ uint64_t xi_desc(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(128u >> 4) << 16) | ((uint64_t)(256u >> 4) << 32) | (1ull << 46);
}
// every wait is bounded: a pipeline bug must end in an error code, not in a hung GPU
__device__ __forceinline__ bool xi_wait(uint32_t bar, uint32_t parity) {
    for (int spin = 0; spin < (1 << 24); ++spin) {
        uint32_t ok;
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return true;
    }
    return false;
}
__device__ __forceinline__ void xi_bulk(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void xi_ld32(uint32_t taddr, int (&v)[32]) {
#pragma unroll
    for (int c0 = 0; c0 < 32; c0 += 16)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                     : "=r"(v[c0]), "=r"(v[c0 + 1]), "=r"(v[c0 + 2]), "=r"(v[c0 + 3]), "=r"(v[c0 + 4]), "=r"(v[c0 + 5]), "=r"(v[c0 + 6]),
                       "=r"(v[c0 + 7]), "=r"(v[c0 + 8]), "=r"(v[c0 + 9]), "=r"(v[c0 + 10]), "=r"(v[c0 + 11]), "=r"(v[c0 + 12]),
                       "=r"(v[c0 + 13]), "=r"(v[c0 + 14]), "=r"(v[c0 + 15])
                     : "r"(taddr + c0));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
// int32 -> fp64 without I2F: 2^52 + (v + 2^31) is exact in the low mantissa word
__device__ __forceinline__ double xi_pow2(int e) { return __hiloint2double((1023 + e) << 20, 0); }
__device__ __forceinline__ double xi_i2d(int v) { return __hiloint2double(0x43300000, v ^ (int)0x80000000) - 4503601774854144.0; }

__device__ __forceinline__ void xi_ld8(uint32_t taddr, int (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr));
}
// the registers of the load are operands of the wait, so that nothing that reads them can be scheduled above it
__device__ __forceinline__ void xi_ld_wait8(int (&v)[8]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(v[0]), "+r"(v[1]), "+r"(v[2]), "+r"(v[3]), "+r"(v[4]), "+r"(v[5]), "+r"(v[6]), "+r"(v[7])
                 :: "memory");
}
// int64 -> fp64 without I2F for |s| < 2^51: 2^52 + 2^51 + s is exact in the mantissa
__device__ __forceinline__ double xi_l2d(long long s) { return __longlong_as_double(s + 0x4338000000000000LL) - 6755399441055744.0; }
// Read-out of the 7 accumulator groups of this thread's row: 32 columns, 8 at a time; for a column the groups are first merged
// EXACTLY in 64-bit integers -- hi = D_0 2^21 + D_1 2^14 + D_2 2^7 + D_3, lo = D_4 2^14 + D_5 2^7 + D_6, |hi| <= N 2^33.1 -- and
// only the two sums go through the FP64 pipe (the read-out is bound by that pipe: 64 FMA / clock / SM),
//   sum_g 2^-(7g+12) D_g = hi 2^-33 + lo 2^-54.
// The next 8-column load is in flight while the current one is merged.  PHASE_B = false: a[j] = that value.  PHASE_B = true:
// p1 += sum_j a[j] b[j], p2 += sum_j an[j] b[j]; b itself is never stored.
template <bool PHASE_B>
__device__ __forceinline__ void xi_readout(uint32_t tbase, double (&a)[32], const double (&an)[32], double& p1, double& p2) {
    static_assert(XI_S == 7, "the hi / lo split below is written for 7 groups");
    int v[2][8];
    xi_ld8(tbase, v[0]);
    double q1a = 0.0, q1b = 0.0, q2a = 0.0, q2b = 0.0;
    const double c_hi = xi_pow2(-33), c_lo = xi_pow2(-54);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        long long hi[8], lo[8];
#pragma unroll
        for (int g = 0; g < XI_S; ++g) {
            const int n = c * XI_S + g;
            xi_ld_wait8(v[n & 1]);
            if (n + 1 < 4 * XI_S) xi_ld8(tbase + (uint32_t)(((n + 1) % XI_S) * 64 + ((n + 1) / XI_S) * 8), v[(n + 1) & 1]);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const long long d = v[n & 1][j];
                if (g == 0) hi[j] = d * (1LL << 21);
                else if (g == 1) hi[j] += d * (1LL << 14);
                else if (g == 2) hi[j] += d * (1LL << 7);
                else if (g == 3) hi[j] += d;
                else if (g == 4) lo[j] = d * (1LL << 14);
                else if (g == 5) lo[j] += d * (1LL << 7);
                else lo[j] += d;
            }
        }
#pragma unroll
        for (int j = 0; j < 8; j += 2) {
            const double b0 = fma(xi_l2d(hi[j]), c_hi, xi_l2d(lo[j]) * c_lo), b1 = fma(xi_l2d(hi[j + 1]), c_hi, xi_l2d(lo[j + 1]) * c_lo);
            if constexpr (PHASE_B) {
                q1a = fma(a[c * 8 + j], b0, q1a); q1b = fma(a[c * 8 + j + 1], b1, q1b);
                q2a = fma(an[c * 8 + j], b0, q2a); q2b = fma(an[c * 8 + j + 1], b1, q2b);
            } else {
                a[c * 8 + j] = b0;
                a[c * 8 + j + 1] = b1;
            }
        }
    }
    if constexpr (PHASE_B) {
        p1 = q1a + q1b;
        p2 = q2a + q2b;
    }
}

// The MMAs of one K block (32 basis functions) of a stage at shared address st: Theta digit s (M = 128 rows) against the operand
// digits t = 0 .. 6 - s.  The operand's digit blocks lie one behind the other in the stage (64 rows each) and group s + t owns TMEM
// columns [64 (s + t), + 64), so ONE instruction with N = 64 cnt covers cnt consecutive t: its B operand is "rows" t0*64 .. of the
// stacked digit blocks, its accumulator the cnt adjacent groups (28 digit products in 10 instructions; kind::i8 instructions
// below N = 128 run at the N = 128 rate).  Nmma = live operand rows rounded up to 16; `first` overwrites the accumulators.
__device__ __forceinline__ void xi_mma_kblock(uint32_t tmem, uint32_t st, uint32_t Nmma, bool first) {
    // instruction descriptor: D = S32 (2 << 4), A = B = signed 8 bit (1 << 7, 1 << 10), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
    const uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((128u >> 4) << 24);
#pragma unroll
    for (int s = 0; s < XI_S; ++s) {
        const uint64_t da = xi_desc(st + s * XI_TH_BLK);
        const uint32_t accum = (first && s == 0) ? 0u : 1u;
#pragma unroll
        for (int t0 = 0; t0 < XI_S - s; t0 += XI_CAT) {
            const int cnt = (XI_S - s - t0) < XI_CAT ? (XI_S - s - t0) : XI_CAT;
            const uint32_t Ni = 64u * (cnt - 1) + Nmma;
            const uint32_t id = idesc | ((Ni >> 3) << 17);
            const uint64_t db = xi_desc(st + XI_TH_STAGE + t0 * XI_F_BLK);
            asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p; }"
                         ::"r"(tmem + (uint32_t)(s + t0) * 64), "l"(da), "l"(db), "r"(id), "r"(accum) : "memory");
        }
    }
}

// CTA set-up shared by the INT8 kernels: mbarriers (full[], empty[], acc_full, acc_empty), 512 TMEM columns; returns the TMEM base
__device__ __forceinline__ uint32_t xi_cta_setup(uint32_t full, uint32_t* tmem_base_s) {
    const uint32_t empty = full + 8 * XI_STAGES, acc_full = empty + 8 * XI_STAGES, acc_empty = acc_full + 8;
    if (threadIdx.x == 0) {
        for (int i = 0; i < XI_STAGES; ++i) { mbar_init(full + 8 * i, 1); mbar_init(empty + 8 * i, 1); }
        mbar_init(acc_full, 1);
        mbar_init(acc_empty, 8);            // one arrival per epilogue warp
        fence_barrier_init();
    }
    if (threadIdx.x < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_s)), "r"((uint32_t)XI_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    return *tmem_base_s;
}

// COUL (lo_set_coulomb_mode(COMPRESSED)): two more phases per item, aJ = U Theta_i and bJ = W Theta_j (Eq. 19/22
// first term, "forming the projected vectors must occur four times"), reduced with the same weights into ejpart.
template <bool COUL>
__global__ void __launch_bounds__(384, 1) k_exchange_i8(const int8_t* __restrict__ Uq, const int8_t* __restrict__ Wq, const int8_t* __restrict__ Thq,
                                                        const double* __restrict__ wq, const double* __restrict__ thScale,
                                                        const ExTile* __restrict__ tiles, long long n_items, int NB, int NBcap, int KB, int Wcap,
                                                        double* __restrict__ ekpart, double* __restrict__ ejpart, int* __restrict__ fail) {
    constexpr int NPH = COUL ? 4 : 2;       // phases of an item: (U, Theta_pj), (W, Theta_pi) [, (U, Theta_pi), (W, Theta_pj)]
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bar_s[2 * XI_STAGES + 2];      // full[], empty[], acc_full, acc_empty
    __shared__ uint32_t tmem_base_s;
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t full = smem_u32(&bar_s[0]), empty = full + 8 * XI_STAGES, acc_full = empty + 8 * XI_STAGES, acc_empty = acc_full + 8;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // partial sums: two rows per CTA (one per column half of the epilogue warps), zeroed here, updated by their owners only
    for (int i = tid; i < 4 * Wcap; i += 384) {
        ekpart[(size_t)blockIdx.x * 4 * Wcap + i] = 0.0;
        if constexpr (COUL) ejpart[(size_t)blockIdx.x * 4 * Wcap + i] = 0.0;
    }
    const uint32_t tmem = xi_cta_setup(full, &tmem_base_s);
    const long long my_items = n_items > (long long)blockIdx.x ? (n_items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    bool ok = true;
    if (warp < 4) {
        reg_dec_producer();
        if (warp == 0 && lane == 0) {
            // ===== feed: per item two phases (a: U with Theta_pj, b: W with Theta_pi), per phase KB stages
            int slot = 0;
            uint32_t phase = 0;
            for (long long it = 0; it < my_items && ok; ++it) {
                const long long q = blockIdx.x + it * gridDim.x;
                const int tile_idx = (int)(q / NB), nb = (int)(q % NB);
                const ExTile tile = tiles[tile_idx];
                if (it + 1 < my_items) {
                    // the factor digits of the next item come from HBM (every tile is read by NB CTAs at about the same time, once
                    // per call): ask L2 for them one item ahead
                    const size_t nxt = (size_t)((q + gridDim.x) / NB) * KB * XI_F_STAGE;
                    for (int kb = 0; kb < KB; ++kb) {
                        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(Uq + nxt + (size_t)kb * XI_F_STAGE), "r"((uint32_t)XI_F_STAGE) : "memory");
                        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(Wq + nxt + (size_t)kb * XI_F_STAGE), "r"((uint32_t)XI_F_STAGE) : "memory");
                    }
                }
                for (int ph = 0; ph < NPH && ok; ++ph) {
                    const int8_t* th = Thq + (size_t)(((ph == 1 || ph == 2) ? tile.pi : tile.pj) * NBcap + nb) * KB * XI_TH_STAGE;
                    const int8_t* fq = ((ph & 1) ? Wq : Uq) + (size_t)tile_idx * KB * XI_F_STAGE;
                    for (int kb = 0; kb < KB; ++kb) {
                        ok = xi_wait(empty + 8 * slot, phase ^ 1);
                        if (!ok) break;
                        const uint32_t st = sbase + slot * XI_STAGE, bar = full + 8 * slot;
                        mbar_expect_tx(bar, XI_STAGE);
                        xi_bulk(st, th + (size_t)kb * XI_TH_STAGE, XI_TH_STAGE, bar);
                        xi_bulk(st + XI_TH_STAGE, fq + (size_t)kb * XI_F_STAGE, XI_F_STAGE, bar);
                        if (++slot == XI_STAGES) { slot = 0; phase ^= 1; }
                    }
                }
            }
            if (!ok) atomicExch(fail, 1);
        } else if (warp == 1 && lane == 0) {
            // ===== MMA issue: 28 digit products per K block, group g = s + t accumulates in TMEM columns [64 g, 64 g + N)
            int slot = 0;
            uint32_t phase = 0, pe = 1;             // the accumulators start out free
            for (long long it = 0; it < my_items && ok; ++it) {
                const long long q = blockIdx.x + it * gridDim.x;
                const ExTile tile = tiles[(int)(q / NB)];
                const uint32_t Nmma = (uint32_t)((tile.nfrag * 8 + 15) / 16) * 16;
                for (int ph = 0; ph < NPH && ok; ++ph) {
                    ok = xi_wait(acc_empty, pe);
                    if (!ok) break;
                    pe ^= 1;
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    for (int kb = 0; kb < KB; ++kb) {
                        ok = xi_wait(full + 8 * slot, phase);
                        if (!ok) break;
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t st = sbase + slot * XI_STAGE;
                        xi_mma_kblock(tmem, st, Nmma, kb == 0);
                        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(empty + 8 * slot) : "memory");
                        if (++slot == XI_STAGES) { slot = 0; phase ^= 1; }
                    }
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(acc_full) : "memory");
                }
            }
            if (!ok) atomicExch(fail, 1);
        }
    } else {
        // ===== epilogue: lane quadrant warp % 4 (walker rows 32 quad .. + 31), column half (warp - 4) / 4 (factor rows 32 half .. + 31)
        reg_inc_consumer();
        const int quad = warp & 3, half = (warp - 4) >> 2;
        const int m = quad * 32 + lane, wl = m >> 1, c = m & 1;       // row of the walker block = 2 wl + c
        const uint32_t tbase = tmem + ((uint32_t)(quad * 32) << 16) + (uint32_t)half * 32;
        double2* mypart = reinterpret_cast<double2*>(ekpart) + (size_t)(2 * blockIdx.x + half) * Wcap;
        double2* mypartJ = COUL ? reinterpret_cast<double2*>(ejpart) + (size_t)(2 * blockIdx.x + half) * Wcap : nullptr;
        uint32_t pf = 0;
        for (long long it = 0; it < my_items && ok; ++it) {
            const long long q = blockIdx.x + it * gridDim.x;
            const int tile_idx = (int)(q / NB), nb = (int)(q % NB);
            const ExTile tile = tiles[tile_idx];
            const int w = nb * 64 + wl, nrow = tile.nfrag * 8 - half * 32;      // live columns of this thread: [0, nrow)
            const double* wrow = wq + tile.row0 + half * 32;
            const double sw = thScale[(size_t)tile.pj * Wcap + w] * thScale[(size_t)tile.pi * Wcap + w];
#pragma unroll 1
            for (int pp = 0; pp < NPH / 2; ++pp) {          // pp = 0: exchange projections, pp = 1: compressed-Coulomb projections
                double a[32], an[32], p1 = 0.0, p2 = 0.0;
                // the weights of this thread's factor rows, fetched before the accumulators are waited for (0 beyond the tile: those
                // TMEM columns were never written)
#pragma unroll
                for (int j = 0; j < 32; ++j) an[j] = j < nrow ? __ldg(wrow + j) : 0.0;
                // ---- first phase of the pair: recombine, weight, fetch the re/im partner row
                ok = xi_wait(acc_full, pf);
                ok = __all_sync(0xffffffffu, ok);
                if (!ok) break;
                pf ^= 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                xi_readout<false>(tbase, a, an, p1, p2);
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(acc_empty);
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    a[j] *= an[j];
                    an[j] = __shfl_xor_sync(0xffffffffu, a[j], 1);
                }
                // ---- second phase: p1 = sum a_own b_own, p2 = sum a_partner b_own
                ok = xi_wait(acc_full, pf);
                ok = __all_sync(0xffffffffu, ok);
                if (!ok) break;
                pf ^= 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                xi_readout<true>(tbase, a, an, p1, p2);
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(acc_empty);
                // row re (c = 0): p1 = sum a_re b_re, p2 = sum a_im b_re;  row im: p1 = sum a_im b_im, p2 = sum a_re b_im
                const double o1 = __shfl_xor_sync(0xffffffffu, p1, 1), o2 = __shfl_xor_sync(0xffffffffu, p2, 1);
                if (c == 0) {
                    double2* dst = (COUL && pp) ? mypartJ : mypart;
                    double2 prev = dst[w];
                    prev.x = fma(sw, p1 - o1, prev.x);
                    prev.y = fma(sw, p2 + o2, prev.y);
                    dst[w] = prev;
                }
            }
        }
        if (!ok && lane == 0) atomicExch(fail, 1);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"((uint32_t)XI_TMEM_COLS) : "memory");
}

// ---- Coulomb / one-body contraction on the same route -------------------------------------------------------------------------
// X^g_w = sum_{o,p} Lbar^g_op Theta_w[p][o] (Eq. 16; row n_chol of Lbar is hbar: the one-body term) from the Theta
// digits of this call and digits of Lbar cut once: Lq [gt][o][kb][7][64 rows x 32 B], rows g = 64 gt .. of Lbar, one power of two
// per (row g, orbital o) segment (eL).  A work item = (64 rows g, block of 64 walkers, split sp of the orbitals).  The Theta rows carry one exponent
// per (orbital, walker), so the int32 accumulators are read out after every orbital (12 K blocks at N = 378) and summed in fp64
// registers with that orbital's scale -- which also keeps every int32 sum far from overflow.  Output: Xpart[sp][g][2 w + c], the
// layout k_ej reads (it adds the split partials, forms E_J and picks the hbar row).
__global__ void __launch_bounds__(384, 1) k_coulomb_i8(const int8_t* __restrict__ Lq, const int8_t* __restrict__ Thq, const int* __restrict__ eL,
                                                       const double* __restrict__ thScale, long long n_items, int NB, int NBcap, int KB, int Wcap,
                                                       int O_tot, int nsplit, int Xp, int ldw, double* __restrict__ Xpart, int* __restrict__ fail) {
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bar_s[2 * XI_STAGES + 2];      // full[], empty[], acc_full, acc_empty
    __shared__ uint32_t tmem_base_s;
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t full = smem_u32(&bar_s[0]), empty = full + 8 * XI_STAGES, acc_full = empty + 8 * XI_STAGES, acc_empty = acc_full + 8;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tmem = xi_cta_setup(full, &tmem_base_s);
    const long long my_items = n_items > (long long)blockIdx.x ? (n_items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    bool ok = true;
    // item q -> (gt, nb, sp), sp fastest: the splits of one (gt, nb) run side by side on neighbouring CTAs
#define XI_CO_ITEM(q_)                                                              \
    const int sp = (int)((q_) % nsplit), nb = (int)(((q_) / nsplit) % NB), gt = (int)((q_) / ((long long)nsplit * NB)); \
    const int o0 = (int)((long long)O_tot * sp / nsplit), o1 = (int)((long long)O_tot * (sp + 1) / nsplit)
    if (warp < 4) {
        reg_dec_producer();
        if (warp == 0 && lane == 0) {
            int slot = 0;
            uint32_t phase = 0;
            for (long long it = 0; it < my_items && ok; ++it) {
                XI_CO_ITEM(blockIdx.x + it * gridDim.x);
                for (int o = o0; o < o1 && ok; ++o) {
                    const int8_t* th = Thq + (size_t)(o * NBcap + nb) * KB * XI_TH_STAGE;
                    const int8_t* lq = Lq + ((size_t)gt * O_tot + o) * KB * XI_F_STAGE;
                    for (int kb = 0; kb < KB; ++kb) {
                        ok = xi_wait(empty + 8 * slot, phase ^ 1);
                        if (!ok) break;
                        const uint32_t st = sbase + slot * XI_STAGE, bar = full + 8 * slot;
                        mbar_expect_tx(bar, XI_STAGE);
                        xi_bulk(st, th + (size_t)kb * XI_TH_STAGE, XI_TH_STAGE, bar);
                        xi_bulk(st + XI_TH_STAGE, lq + (size_t)kb * XI_F_STAGE, XI_F_STAGE, bar);
                        if (++slot == XI_STAGES) { slot = 0; phase ^= 1; }
                    }
                }
            }
            if (!ok) atomicExch(fail, 1);
        } else if (warp == 1 && lane == 0) {
            int slot = 0;
            uint32_t phase = 0, pe = 1;
            for (long long it = 0; it < my_items && ok; ++it) {
                XI_CO_ITEM(blockIdx.x + it * gridDim.x);
                (void)nb; (void)gt;
                for (int o = o0; o < o1 && ok; ++o) {
                    ok = xi_wait(acc_empty, pe);
                    if (!ok) break;
                    pe ^= 1;
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    for (int kb = 0; kb < KB; ++kb) {
                        ok = xi_wait(full + 8 * slot, phase);
                        if (!ok) break;
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        xi_mma_kblock(tmem, sbase + slot * XI_STAGE, 64u, kb == 0);
                        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(empty + 8 * slot) : "memory");
                        if (++slot == XI_STAGES) { slot = 0; phase ^= 1; }
                    }
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(acc_full) : "memory");
                }
            }
            if (!ok) atomicExch(fail, 1);
        }
    } else {
        reg_inc_consumer();
        const int quad = warp & 3, half = (warp - 4) >> 2;
        const int m = quad * 32 + lane;                                // row of the walker block = 2 (w % 64) + c
        const uint32_t tbase = tmem + ((uint32_t)(quad * 32) << 16) + (uint32_t)half * 32;
        uint32_t pf = 0;
        for (long long it = 0; it < my_items && ok; ++it) {
            XI_CO_ITEM(blockIdx.x + it * gridDim.x);
            const int w = nb * 64 + (m >> 1), g0 = gt * 64 + half * 32;
            double x[32], b[32], d1 = 0.0, d2 = 0.0;
#pragma unroll
            for (int j = 0; j < 32; ++j) x[j] = 0.0;
            for (int o = o0; o < o1; ++o) {
                const double sw = thScale[(size_t)o * Wcap + w];
                ok = xi_wait(acc_full, pf);
                ok = __all_sync(0xffffffffu, ok);
                if (!ok) break;
                pf ^= 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                xi_readout<false>(tbase, b, b, d1, d2);
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(acc_empty);
                const int* el = eL + (size_t)o * Xp + g0;        // the same 128 bytes for every lane: one broadcast line
#pragma unroll
                for (int j = 0; j < 32; ++j) x[j] = fma(b[j] * xi_pow2(__ldg(el + j)), sw, x[j]);
            }
            if (!ok) break;
            // a warp stores 32 consecutive doubles of one row g per j: coalesced
            double* out = Xpart + ((size_t)sp * Xp + g0) * ldw + (size_t)nb * 128 + m;
#pragma unroll
            for (int j = 0; j < 32; ++j) out[(size_t)j * ldw] = x[j];
        }
        if (!ok && lane == 0) atomicExch(fail, 1);
    }
#undef XI_CO_ITEM
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"((uint32_t)XI_TMEM_COLS) : "memory");
}

// Lbar -> exponents eL[o][g] of every (row g, orbital o) segment (one warp each: a localized orbital far from the site of g holds
// much smaller entries than the row's largest, and the accumulators are read out per orbital anyway) and digits
// Lq [gt][o][kb][7][64 x 32].
__global__ void __launch_bounds__(256) k_lbar_exponents(const double* __restrict__ Lbar, int* __restrict__ eL, int Xp, int O_tot, int N_pad) {
    const int lane = threadIdx.x & 31;
    const long long seg = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (seg >= (long long)Xp * O_tot) return;
    const int g = (int)(seg / O_tot), o = (int)(seg % O_tot);
    const double* src = Lbar + (size_t)seg * N_pad;
    double mx = 0.0;
    for (int i = lane; i < N_pad; i += 32) mx = fmax(mx, fabs(src[i]));
#pragma unroll
    for (int d = 16; d; d >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    if (lane == 0) eL[(size_t)o * Xp + g] = row_exponent(mx);
}
__global__ void __launch_bounds__(256) k_slice_lbar(const double* __restrict__ Lbar, const int* __restrict__ eL, int8_t* __restrict__ Lq, int O_tot,
                                                    int N_pad, int KB, int Xp) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, gt = blockIdx.x, o = blockIdx.y;
    const int nch = 2 * KB;
    int8_t* blk = Lq + ((size_t)gt * O_tot + o) * KB * XI_F_STAGE;
    for (int r = warp; r < 64; r += 8) {
        const int g = gt * 64 + r;
        const double* src = Lbar + ((size_t)g * O_tot + o) * N_pad;
        const double inv = scalbn(1.0, -eL[(size_t)o * Xp + g]);
        for (int ch = lane; ch < nch; ch += 32) {
            const int k0 = ch * 16;
            int4 out[XI_S];
            if (k0 < N_pad) slice16(src + k0, inv, out);
            else {
#pragma unroll
                for (int s = 0; s < XI_S; ++s) out[s] = make_int4(0, 0, 0, 0);
            }
            int8_t* dst = blk + (size_t)(ch >> 1) * XI_F_STAGE + (r >> 3) * 256 + (ch & 1) * 128 + (r & 7) * 16;
#pragma unroll
            for (int s = 0; s < XI_S; ++s) *reinterpret_cast<int4*>(dst + s * XI_F_BLK) = out[s];
        }
    }
}

// a bounded wait expired somewhere: poison the partial sums so that every energy of the call comes out NaN
__global__ void k_i8_poison(const int* __restrict__ fail, double* __restrict__ ekpart, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (*fail && i < n) ekpart[i] = __longlong_as_double(0x7ff8000000000000LL);
}

}  // namespace

void free_exchange_i8(lo_factors* f) {
    void* ptrs[] = {f->dUq, f->dWq, f->dThq, f->dWgtQ, f->dThScale, f->dEKq, f->dEJq, f->dI8Fail, f->dLq, f->dELq, f->dLtq, f->dELt, f->dXq, f->dXScale};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    f->dUq = f->dWq = f->dThq = f->dLq = nullptr;
    f->dELq = f->dELt = nullptr;
    f->dLtq = f->dXq = nullptr;
    f->dXScale = nullptr;
    f->dWgtQ = f->dThScale = f->dEKq = f->dEJq = nullptr;
    f->dI8Fail = nullptr;
    f->i8_bytes = 0;
}

// Slices the packed factor rows once (Uq, Wq, wq) and allocates the per-call buffers (Thq, thScale, partial sums).
lo_status build_exchange_i8(lo_factors* f) {
#define CK(call)                                                                                                         \
    do {                                                                                                                 \
        cudaError_t e_ = (call);                                                                                         \
        if (e_ != cudaSuccess) {                                                                                         \
            set_error(std::string("lo_set_exchange_mode: ") + #call + ": " + cudaGetErrorString(e_));                    \
            free_exchange_i8(f);                                                                                         \
            return e_ == cudaErrorMemoryAllocation ? LO_ENOMEM : LO_ECUDA;                                               \
        }                                                                                                                \
    } while (0)
    if (f->dUq) return LO_OK;
    CK(cudaSetDevice(f->device));
    static bool configured = false;
    if (!configured) {
        CK(cudaFuncSetAttribute(k_exchange_i8<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, XI_SMEM));
        CK(cudaFuncSetAttribute(k_exchange_i8<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, XI_SMEM));
        CK(cudaFuncSetAttribute(k_coulomb_i8, cudaFuncAttributeMaxDynamicSharedMemorySize, XI_SMEM));
        configured = true;
    }
    const int KB = (f->N_pad + 31) / 32, NBcap = f->Wcap / 64;
    const size_t fq_bytes = (size_t)std::max<long long>(f->n_tiles, 1) * KB * XI_F_STAGE;
    const size_t th_bytes = (size_t)f->O_tot * NBcap * KB * XI_TH_STAGE;
    const long long rows_al = f->rows + 64;
    int *eU = nullptr, *eW = nullptr;
    CK(cudaMalloc(&f->dUq, fq_bytes));
    CK(cudaMalloc(&f->dWq, fq_bytes));
    CK(cudaMalloc(&f->dThq, th_bytes));
    CK(cudaMalloc(&f->dWgtQ, (size_t)rows_al * 8));
    CK(cudaMalloc(&f->dThScale, (size_t)f->O_tot * f->Wcap * 8));
    CK(cudaMalloc(&f->dEKq, (size_t)2 * f->num_sms * f->Wcap * 16));
    CK(cudaMalloc(&f->dEJq, (size_t)2 * f->num_sms * f->Wcap * 16));
    const size_t lq_bytes = (size_t)(f->Xp / 64) * f->O_tot * KB * XI_F_STAGE;
    CK(cudaMalloc(&f->dLq, lq_bytes));
    CK(cudaMalloc(&f->dELq, (size_t)f->Xp * f->O_tot * 4));
    CK(cudaMalloc(&f->dI8Fail, 4));
    CK(cudaMemset(f->dI8Fail, 0, 4));
    CK(cudaMemset(f->dWgtQ, 0, (size_t)rows_al * 8));
    CK(cudaMemset(f->dThq, 0, th_bytes));
    f->i8_bytes = 2 * fq_bytes + th_bytes + lq_bytes + (size_t)rows_al * 8;
    {
        // digits of Lbar (rows g, incl. the hbar row) for the Coulomb / one-body contraction
        k_lbar_exponents<<<(unsigned)(((long long)f->Xp * f->O_tot + 7) / 8), 256>>>(f->ops->dLbar, f->dELq, f->Xp, f->O_tot, f->N_pad);
        dim3 gl(f->Xp / 64, f->O_tot);
        k_slice_lbar<<<gl, 256>>>(f->ops->dLbar, f->dELq, f->dLq, f->O_tot, f->N_pad, KB, f->Xp);
        CK(cudaDeviceSynchronize());
    }
    if (f->ops->dLt) {
        // propagator (LO_SETUP_PROPAGATOR): digits of Lt [r(p,q)][g] (one exponent per row) and room for the digits of the fields
        const int KBx = (f->ops->Xk_pad + 31) / 32;
        const size_t ltq_bytes = (size_t)(f->ops->tri_pad / 64) * KBx * XI_F_STAGE, xq_bytes = (size_t)NBcap * KBx * XI_TH_STAGE;
        CK(cudaMalloc(&f->dLtq, ltq_bytes));
        CK(cudaMalloc(&f->dELt, (size_t)f->ops->tri_pad * 4));
        CK(cudaMalloc(&f->dXq, xq_bytes));
        CK(cudaMalloc(&f->dXScale, (size_t)f->Wcap * 8));
        CK(cudaMemset(f->dXq, 0, xq_bytes));
        f->i8_bytes += ltq_bytes + xq_bytes;
        k_lbar_exponents<<<(unsigned)((f->ops->tri_pad + 7) / 8), 256>>>(f->ops->dLt, f->dELt, (int)f->ops->tri_pad, 1, f->ops->Xk_pad);
        dim3 gl((unsigned)(f->ops->tri_pad / 64), 1);
        k_slice_lbar<<<gl, 256>>>(f->ops->dLt, f->dELt, f->dLtq, 1, f->ops->Xk_pad, KBx, (int)f->ops->tri_pad);
        CK(cudaDeviceSynchronize());
    }
    if (f->n_tiles > 0) {
        cudaError_t e1 = cudaMalloc(&eU, (size_t)rows_al * 4), e2 = cudaMalloc(&eW, (size_t)rows_al * 4);
        if (e1 != cudaSuccess || e2 != cudaSuccess) {
            cudaFree(eU); cudaFree(eW);
            (void)cudaGetLastError();
            free_exchange_i8(f);
            set_error("lo_set_exchange_mode: out of device memory for the slicing scratch");
            return LO_ENOMEM;
        }
        cudaMemset(eU, 0, (size_t)rows_al * 4);
        cudaMemset(eW, 0, (size_t)rows_al * 4);
        k_slice_factors<<<(unsigned)f->n_tiles, 256>>>(f->dU, f->dTiles, f->dUq, eU, f->N_pad, KB);
        k_slice_factors<<<(unsigned)f->n_tiles, 256>>>(f->dW, f->dTiles, f->dWq, eW, f->N_pad, KB);
        k_i8_weights<<<(unsigned)((f->rows + 255) / 256), 256>>>(f->dWgt, eU, eW, f->dWgtQ, f->rows);
        cudaError_t e = cudaDeviceSynchronize();
        cudaFree(eU); cudaFree(eW);
        CK(e);
    }
    return LO_OK;
#undef CK
}

// INT8 route, per call: digits of the Theta^T panels (used by the Coulomb and the exchange kernels of this call)
void launch_slice_theta_i8(lo_factors* f, int n_w, cudaStream_t stream) {
    const int KB = (f->N_pad + 31) / 32, NBcap = f->Wcap / 64, NB = (n_w + 63) / 64, n_wpad = NB * 64;
    const long long warps = (long long)f->O_tot * n_wpad;
    k_slice_theta<<<(unsigned)((warps + 7) / 8), 256, 0, stream>>>(f->dThT, f->dThq, f->dThScale, f->O_tot, f->ldw, f->N_pad, KB, NBcap, f->Wcap, n_wpad);
}

// S2 + S3 on the INT8 route: X^g_w into f->dXpart as `nsplit` (returned) split partials over the orbitals; the caller runs k_ej
int launch_coulomb_i8(lo_factors* f, int n_w, cudaStream_t stream) {
    const int KB = (f->N_pad + 31) / 32, NBcap = f->Wcap / 64, NB = (n_w + 63) / 64;
    const long long base = (long long)(f->Xp / 64) * NB;
    int nsplit = 1;
    double best = -1.0;
    for (int s = 1; s <= std::min(MAX_SPLIT, f->O_tot); ++s) {       // fill the last wave
        const long long items = base * s, waves = (items + f->num_sms - 1) / f->num_sms;
        const double eff = (double)items / (double)(waves * f->num_sms);
        if (eff > best + 0.02) { best = eff; nsplit = s; }
    }
    const long long items = base * nsplit;
    const int grid = (int)std::min<long long>(items, f->num_sms);
    k_coulomb_i8<<<grid, 384, XI_SMEM, stream>>>(f->dLq, f->dThq, f->dELq, f->dThScale, items, NB, NBcap, KB, f->Wcap, f->O_tot, nsplit, f->Xp, f->ldw,
                                                 f->dXpart, f->dI8Fail);
    return nsplit;
}

// Propagator formation B[r(p,q)][w] = sum_g L^g_pq x^g_w on the INT8 route: the packed fields f->dXT ([2w + c][g],
// the layout of a one-orbital Theta^T panel with K = g) are cut into digits like Theta, the GEMM is k_coulomb_i8 with one
// "orbital" segment of ceil(n_chol / 32) K blocks against the digits of Lt; output straight into f->dB.
void launch_propagator_i8(lo_factors* f, int n_w, cudaStream_t stream) {
    const int KBx = (f->ops->Xk_pad + 31) / 32, NBcap = f->Wcap / 64, NB = (n_w + 63) / 64, n_wpad = NB * 64;
    k_slice_theta<<<(unsigned)((n_wpad + 7) / 8), 256, 0, stream>>>(f->dXT, f->dXq, f->dXScale, 1, f->ldw, f->ops->Xk_pad, KBx, NBcap, f->Wcap, n_wpad);
    const long long items = (long long)(f->ops->tri_pad / 64) * NB;
    const int grid = (int)std::min<long long>(items, f->num_sms);
    k_coulomb_i8<<<grid, 384, XI_SMEM, stream>>>(f->dLtq, f->dXq, f->dELt, f->dXScale, items, NB, NBcap, KBx, f->Wcap, 1, 1, (int)f->ops->tri_pad, f->ldw,
                                                 f->dB, f->dI8Fail);
    k_i8_poison<<<(f->ldw + 255) / 256, 256, 0, stream>>>(f->dI8Fail, f->dB, f->ldw);      // an expired wait: NaN in row 0 of every walker
}

// S4 on the INT8 route (the Theta digits of this call are in place: launch_slice_theta_i8); the partial sums land in f->dEKq as
// 2 * grid rows (*n_part) for k_finalize.
void launch_exchange_i8(lo_factors* f, int n_w, cudaStream_t stream, bool coul, const double** part, int* n_part, const double** partJ) {
    const int KB = (f->N_pad + 31) / 32, NBcap = f->Wcap / 64, NB = (n_w + 63) / 64;
    const long long items = f->n_tiles * NB;
    const int grid = (int)std::min<long long>(std::max<long long>(items, 1), f->num_sms);
    if (coul)
        k_exchange_i8<true><<<grid, 384, XI_SMEM, stream>>>(f->dUq, f->dWq, f->dThq, f->dWgtQ, f->dThScale, f->dTiles, items, NB, NBcap, KB, f->Wcap, f->dEKq,
                                                            f->dEJq, f->dI8Fail);
    else
        k_exchange_i8<false><<<grid, 384, XI_SMEM, stream>>>(f->dUq, f->dWq, f->dThq, f->dWgtQ, f->dThScale, f->dTiles, items, NB, NBcap, KB, f->Wcap, f->dEKq,
                                                             nullptr, f->dI8Fail);
    const int n = grid * 4 * f->Wcap;
    k_i8_poison<<<(n + 255) / 256, 256, 0, stream>>>(f->dI8Fail, f->dEKq, n);
    *part = f->dEKq;
    *n_part = 2 * grid;
    *partJ = coul ? f->dEJq : nullptr;
}

}  // namespace lo
