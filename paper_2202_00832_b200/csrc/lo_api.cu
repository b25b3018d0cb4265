// lo_api.cu -- C ABI entry points of liblo_afqmc.so and the host side of lo_setup
// (half-rotation PAPER.md:127, pair blocks PAPER.md:133, SVD + truncation Eq. 18, rank sort, padding, packing).
#include <omp.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "lo_internal.h"

namespace lo {

std::string& err_buf() {
    static thread_local std::string s;
    return s;
}
void set_error(const std::string& s) { err_buf() = s; }

SharedOps::~SharedOps() {
    if (device >= 0) {
        cudaSetDevice(device);
        if (dLbar) cudaFree(dLbar);
        if (dLt) cudaFree(dLt);
        for (int s = 0; s < 2; ++s)
            if (dPsi[s]) cudaFree(dPsi[s]);
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                 CUtensorMapFloatOOBfill);

lo_status make_tmap(CUtensorMap* tm, const void* base, unsigned long long inner, unsigned long long rows, unsigned box_rows) {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !p) {
            set_error("cuTensorMapEncodeTiled is not available from the driver");
            return LO_ECUDA;
        }
        fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    cuuint64_t dims[2] = {inner, rows};
    cuuint64_t strides[1] = {inner * 8};
    cuuint32_t box[2] = {(cuuint32_t)KTILE, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r));
        return LO_ECUDA;
    }
    return LO_OK;
}

namespace {

#define CK(call)                                                                                          \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess) {                                                                          \
            set_error(std::string(#call) + ": " + cudaGetErrorString(e_));                                \
            return (e_ == cudaErrorMemoryAllocation) ? LO_ENOMEM : LO_ECUDA;                              \
        }                                                                                                 \
    } while (0)

inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

// ---- host half-rotation: Lbar[g][o][p] = sum_q L[g][p][q] psi_s[q][i], hbar[o][p] = sum_q psi[q][i] h[q][p]  (row n_chol)
void host_half_rotate(int N, int n_chol, int n_spin, const int* n_occ, const int* o_base, int O_tot, const double* h, const double* L,
                      const double* const* psi, std::vector<double>& out) {
    out.assign((size_t)(n_chol + 1) * O_tot * N, 0.0);
#pragma omp parallel
    {
        std::vector<double> row(O_tot);
#pragma omp for schedule(static)
        for (int g = 0; g <= n_chol; ++g) {
            const double* M = (g < n_chol) ? L + (size_t)g * N * N : h;
            double* dst = out.data() + (size_t)g * O_tot * N;
            for (int p = 0; p < N; ++p) {
                std::fill(row.begin(), row.end(), 0.0);
                const double* mp = M + (size_t)p * N;   // symmetric: row p == column p
                for (int q = 0; q < N; ++q) {
                    const double a = mp[q];
                    for (int s = 0; s < n_spin; ++s) {
                        const double* ps = psi[s] + (size_t)q * n_occ[s];
                        double* r = row.data() + o_base[s];
                        for (int i = 0; i < n_occ[s]; ++i) r[i] += a * ps[i];
                    }
                }
                for (int o = 0; o < O_tot; ++o) dst[(size_t)o * N + p] = row[o];
            }
        }
    }
}

// ---- host pair block: Y[q][p] layout chosen so that row q of `G` is COLUMN q of Y^{ij}:  G[q][p] = Y^{ij}_pq
void host_pair_gram_t(int N, int n_chol, int O_tot, const double* Lbar, int oi, int oj, double* G) {
    std::fill(G, G + (size_t)N * N, 0.0);
    for (int g = 0; g < n_chol; ++g) {
        const double* li = Lbar + ((size_t)g * O_tot + oi) * N;
        const double* lj = Lbar + ((size_t)g * O_tot + oj) * N;
        for (int q = 0; q < N; ++q) {
            const double b = lj[q];
            double* row = G + (size_t)q * N;
            for (int p = 0; p < N; ++p) row[p] += b * li[p];
        }
    }
}

struct PairRec {
    int spin, i, j, r;
    int x;            // index of the pair inside the batch being packed (source of its rows)
    long long src;    // lo_retruncate: first packed row of the pair in the source factor set
    double snext;     // first discarded singular value (0 if none)
};

inline size_t pair_index(int O, int i, int j) { return (size_t)i * O - (size_t)i * (i - 1) / 2 + (j - i); }

// Pair order of the packed arrays: L2 blocks of BO x BO orbitals (row-major over (spin, i-block, j-block)) so that
// the Theta panels a block touches (2*BO panels of ldw*N_pad*8 bytes) stay in the 126 MB L2 while the block's factor
// rows stream through once; inside a block pairs are sorted by rank, descending (done when the ranks are known).
// Returns the pairs in that order and the start index of every block (+ end sentinel).
void enumerate_blocks(const lo_factors* f, std::vector<PairRec>& pairs, std::vector<size_t>& block_start) {
    const double panel_bytes = (double)f->ldw * f->N_pad * 8.0;
    const int BO = std::max(1, std::min(16, (int)(48e6 / (2.0 * panel_bytes))));
    pairs.clear();
    block_start.clear();
    for (int s = 0; s < f->n_spin; ++s) {
        const int O = f->n_occ[s], nb = (O + BO - 1) / BO;
        for (int ib = 0; ib < nb; ++ib)
            for (int jb = ib; jb < nb; ++jb) {
                block_start.push_back(pairs.size());
                for (int i = ib * BO; i < std::min(O, (ib + 1) * BO); ++i)
                    for (int j = std::max(i, jb * BO); j < std::min(O, (jb + 1) * BO); ++j) pairs.push_back({s, i, j, 0, 0, 0, 0.0});
            }
    }
    block_start.push_back(pairs.size());
}

// Appends pairs (ranks known) to the packed layout: sorts [first,last) by rank inside the block, assigns padded row
// offsets, cuts row tiles, appends the weights  -cK m_ij sigma_K  (sig(pr, K) gives sigma_K) and fills `table` with the
// row copies to perform (src_row is set by the caller's src_row_of).
template <class SigmaFn, class SrcFn>
void layout_block(lo_factors* f, PairRec* first, PairRec* last, SigmaFn sig, SrcFn src_row_of, std::vector<GatherRec>& table) {
    std::stable_sort(first, last, [](const PairRec& a, const PairRec& b) { return a.r > b.r; });
    const double cK = f->n_spin == 1 ? 1.0 : 0.5;
    for (PairRec* pr = first; pr != last; ++pr) {
        const size_t k = pair_index(f->n_occ[pr->spin], pr->i, pr->j);
        f->rank[pr->spin][k] = pr->r;
        f->row_off[pr->spin][k] = f->rows;
        f->sigma_next[pr->spin][k] = pr->snext;
        const int r_pad = round_up(pr->r, 8);
        if (r_pad == 0) continue;
        const int F = r_pad / 8, nt = (F + 7) / 8;
        int done = 0;
        for (int t = 0; t < nt; ++t) {
            const int nf = F / nt + (t < F % nt ? 1 : 0);
            ExTile T;
            T.row0 = (int)(f->rows + (long long)done * 8);
            T.nfrag = nf;
            T.pi = f->o_base[pr->spin] + pr->i;
            T.pj = f->o_base[pr->spin] + pr->j;
            f->hTiles.push_back(T);
            done += nf;
        }
        for (int d4 = 0, nt4 = (F + 3) / 4, t = 0; t < nt4; ++t) {      // NEXT-3 cut: <= 4 fragments per tile
            const int nf = F / nt4 + (t < F % nt4 ? 1 : 0);
            ExTile T;
            T.row0 = (int)(f->rows + (long long)d4 * 8);
            T.nfrag = nf;
            T.pi = f->o_base[pr->spin] + pr->i;
            T.pj = f->o_base[pr->spin] + pr->j;
            f->hTiles4.push_back(T);
            d4 += nf;
        }
        const double m = pr->i == pr->j ? 1.0 : 2.0;
        f->hWgt.resize((size_t)f->rows + r_pad, 0.0);
        for (int K = 0; K < pr->r; ++K) f->hWgt[(size_t)f->rows + K] = -cK * m * sig(*pr, K);
        table.push_back({src_row_of(*pr), f->rows, pr->r, 0});
        f->rows += r_pad;
    }
}

lo_status begin_pack(lo_factors* f) {
    for (int s = 0; s < f->n_spin; ++s) {
        const size_t np = (size_t)f->n_occ[s] * (f->n_occ[s] + 1) / 2;
        f->rank[s].assign(np, 0);
        f->row_off[s].assign(np, 0);
        f->sigma_next[s].assign(np, 0.0);
    }
    f->rows = 0;
    f->hTiles.clear();
    f->hTiles4.clear();
    f->hWgt.clear();
    if (f->device >= 0) {
        CK(cudaSetDevice(f->device));
        size_t max_rows = EX_BM;
        for (int s = 0; s < f->n_spin; ++s) max_rows += (size_t)f->n_occ[s] * (f->n_occ[s] + 1) / 2 * round_up(f->N, 8);
        lo_status st = f->bU.reserve(f->device, max_rows * f->N_pad * 8);
        if (st == LO_OK) st = f->bW.reserve(f->device, max_rows * f->N_pad * 8);
        if (st != LO_OK) return st;
        f->dU = static_cast<double*>(f->bU.base);
        f->dW = static_cast<double*>(f->bW.base);
    }
    return LO_OK;
}

// make rows [0, rows + EX_BM) of the packed arrays usable (zero-filled where new)
lo_status grow_pack(lo_factors* f) {
    const size_t bytes = ((size_t)f->rows + EX_BM) * f->N_pad * 8;
    if (f->device >= 0) {
        lo_status st = f->bU.ensure(bytes);
        if (st == LO_OK) st = f->bW.ensure(bytes);
        return st;
    }
    f->hU.resize(bytes / 8, 0.0);
    f->hW.resize(bytes / 8, 0.0);
    return LO_OK;
}

lo_status alloc_workspace(lo_factors* f);

lo_status finish_pack(lo_factors* f) {
    lo_status st = grow_pack(f);
    if (st != LO_OK) return st;
    const size_t rows_alloc = (size_t)f->rows + EX_BM;
    f->hWgt.resize(rows_alloc, 0.0);
    f->n_tiles = (long long)f->hTiles.size();
    f->n_tiles4 = (long long)f->hTiles4.size();
    f->factor_bytes = 2 * rows_alloc * f->N_pad * 8 + rows_alloc * 8 + f->hTiles.size() * sizeof(ExTile);
    if (f->device < 0) return LO_OK;
    CK(cudaSetDevice(f->device));
    CK(cudaMalloc(&f->dWgt, rows_alloc * 8));
    CK(cudaMalloc(&f->dTiles, std::max<size_t>(1, f->hTiles.size()) * sizeof(ExTile)));
    CK(cudaMemcpy(f->dWgt, f->hWgt.data(), rows_alloc * 8, cudaMemcpyHostToDevice));
    if (!f->hTiles.empty()) CK(cudaMemcpy(f->dTiles, f->hTiles.data(), f->hTiles.size() * sizeof(ExTile), cudaMemcpyHostToDevice));
    CK(cudaMalloc(&f->dTiles4, std::max<size_t>(1, f->hTiles4.size()) * sizeof(ExTile)));
    if (!f->hTiles4.empty()) CK(cudaMemcpy(f->dTiles4, f->hTiles4.data(), f->hTiles4.size() * sizeof(ExTile), cudaMemcpyHostToDevice));
    {
        // Static schedule for small problems (a CTA then gets only a handful of items): tiles dealt to num_sms CTAs by
        // accumulated weight, heaviest first to the least loaded CTA (LPT); weight = fragments + 1/2 (per-item overhead);
        // every CTA's list in ascending tile order.  Fixed for the factor set: results stay repeatable.
        const int G = std::max(1, f->num_sms);
        const size_t nt = f->hTiles.size();
        std::vector<int> ord(nt), owner(nt), off(G + 1, 0), lst(nt);
        std::iota(ord.begin(), ord.end(), 0);
        std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return f->hTiles[a].nfrag > f->hTiles[b].nfrag; });
        std::vector<std::pair<double, int>> heap;          // (load, cta) min-heap
        for (int c = 0; c < G; ++c) heap.push_back({0.0, c});
        auto cmp = [](const std::pair<double, int>& a, const std::pair<double, int>& b) { return a.first != b.first ? a.first > b.first : a.second > b.second; };
        std::make_heap(heap.begin(), heap.end(), cmp);
        for (int t : ord) {
            std::pop_heap(heap.begin(), heap.end(), cmp);
            heap.back().first += f->hTiles[t].nfrag + 0.5;
            owner[t] = heap.back().second;
            std::push_heap(heap.begin(), heap.end(), cmp);
        }
        for (size_t t = 0; t < nt; ++t) ++off[owner[t] + 1];
        for (int c = 0; c < G; ++c) off[c + 1] += off[c];
        std::vector<int> pos(off.begin(), off.end() - 1);
        for (size_t t = 0; t < nt; ++t) lst[pos[owner[t]]++] = (int)t;
        CK(cudaMalloc(&f->dSchedOff, (size_t)(G + 1) * 4));
        CK(cudaMalloc(&f->dSchedTile, std::max<size_t>(nt, 1) * 4));
        CK(cudaMemcpy(f->dSchedOff, off.data(), (size_t)(G + 1) * 4, cudaMemcpyHostToDevice));
        if (nt) CK(cudaMemcpy(f->dSchedTile, lst.data(), nt * 4, cudaMemcpyHostToDevice));
    }
    st = make_tmap(&f->tmU, f->dU, f->N_pad, rows_alloc, EX_BM);
    if (st == LO_OK) st = make_tmap(&f->tmW, f->dW, f->N_pad, rows_alloc, EX_BM);
    if (st == LO_OK) st = make_tmap(&f->tmU8, f->dU, f->N_pad, rows_alloc, 8);
    if (st == LO_OK) st = make_tmap(&f->tmW8, f->dW, f->N_pad, rows_alloc, 8);
    for (int k = 0; k < 8 && st == LO_OK; ++k) {
        st = make_tmap(&f->tmUf.m[k], f->dU, f->N_pad, rows_alloc, 8 * (k + 1));
        if (st == LO_OK) st = make_tmap(&f->tmWf.m[k], f->dW, f->N_pad, rows_alloc, 8 * (k + 1));
    }
    if (st != LO_OK) return st;
    return alloc_workspace(f);
}

lo_status alloc_workspace(lo_factors* f) {
    CK(cudaSetDevice(f->device));
    const size_t Wcap = f->Wcap, ldw = f->ldw;
    size_t total = 0;
    auto al = [&](void** p, size_t bytes) -> cudaError_t {
        total += bytes;
        cudaError_t e = cudaMalloc(p, bytes);
        if (e == cudaSuccess) e = cudaMemset(*p, 0, bytes);
        return e;
    };
    CK(al((void**)&f->dThT, (size_t)f->O_tot * ldw * f->N_pad * 8));
    for (int s = 0; s < f->n_spin; ++s) {
        CK(al((void**)&f->dA[s], Wcap * f->n_occ[s] * f->n_occ[s] * 16));
        CK(al((void**)&f->dPhi[s], Wcap * f->N * f->n_occ[s] * 16));
    }
    CK(al((void**)&f->dXpart, (size_t)MAX_SPLIT * f->Xp * ldw * 8));
    CK(al((void**)&f->dEJpart, (size_t)(f->Xp / CO_BM + 1) * Wcap * 16));
    CK(al((void**)&f->dEKpart, (size_t)f->num_sms * Wcap * 16));
    CK(al((void**)&f->dEJLpart, (size_t)f->num_sms * Wcap * 16));
    CK(al((void**)&f->dStatus, 2 * Wcap * 4));
    CK(al((void**)&f->dEout, Wcap * 4 * 16));
    CK(al((void**)&f->dStatusOut, Wcap * 4));
    if (f->ops->dLt) {
        CK(al((void**)&f->dXT, ldw * (size_t)f->ops->Xk_pad * 8));
        CK(al((void**)&f->dB, (size_t)f->ops->tri_pad * ldw * 8));
    }
    f->workspace_bytes = total;
    CK(cudaStreamCreateWithFlags(&f->copyStream, cudaStreamNonBlocking));
    for (int c = 0; c < LO_HOST_CHUNKS; ++c) CK(cudaEventCreateWithFlags(&f->evCopy[c], cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&f->evEnter, cudaEventDisableTiming));
    lo_status st = make_tmap(&f->tmTheta, f->dThT, f->N_pad, (unsigned long long)f->O_tot * ldw, 128);
    if (st == LO_OK) st = make_tmap(&f->tmTheta32, f->dThT, f->N_pad, (unsigned long long)f->O_tot * ldw, 32);
    if (st == LO_OK && f->dXT) st = make_tmap(&f->tmXT, f->dXT, (unsigned long long)f->ops->Xk_pad, ldw, 128);
    if (st != LO_OK) return st;
    return configure_kernels();
}

lo_status upload_lbar(lo_factors* f) {
    SharedOps& ops = *f->ops;
    CK(cudaSetDevice(f->device));
    const size_t K = (size_t)f->O_tot * f->N_pad;
    CK(cudaMalloc(&ops.dLbar, (size_t)f->Xp * K * 8));
    CK(cudaMemset(ops.dLbar, 0, (size_t)f->Xp * K * 8));
    // host [g][o][N] -> device [g][o][N_pad]
    CK(cudaMemcpy2D(ops.dLbar, (size_t)f->N_pad * 8, ops.hLbar.data(), (size_t)f->N * 8, (size_t)f->N * 8,
                    (size_t)(f->n_chol + 1) * f->O_tot, cudaMemcpyHostToDevice));
    f->lbar_bytes = (size_t)f->Xp * K * 8;
    return make_tmap(&ops.tmLbar, ops.dLbar, K, f->Xp, CO_BM);
}

// Propagator operand: Lt[r(p,q)][g] = L^g_pq, p<=q, K-major with g fastest; built on the host in
// row blocks (OpenMP over rows) and uploaded block by block.
lo_status upload_lt(lo_factors* f, const double* L) {
    SharedOps& ops = *f->ops;
    CK(cudaSetDevice(f->device));
    const long long N = f->N;
    ops.tri = N * (N + 1) / 2;
    ops.tri_pad = (ops.tri + CO_BM - 1) / CO_BM * CO_BM;
    ops.Xk_pad = round_up(f->n_chol, KTILE);
    const size_t ld = (size_t)ops.Xk_pad;
    CK(cudaMalloc(&ops.dLt, (size_t)ops.tri_pad * ld * 8));
    CK(cudaMemset(ops.dLt, 0, (size_t)ops.tri_pad * ld * 8));
    const long long RBLK = 8192;
    std::vector<double> buf((size_t)RBLK * ld, 0.0);
    std::vector<int> rp((size_t)ops.tri), rq((size_t)ops.tri);
    {
        long long r = 0;
        for (int p = 0; p < N; ++p)
            for (int q = p; q < N; ++q, ++r) { rp[r] = p; rq[r] = q; }
    }
    for (long long r0 = 0; r0 < ops.tri; r0 += RBLK) {
        const long long nr = std::min(RBLK, ops.tri - r0);
#pragma omp parallel for schedule(static)
        for (long long rr = 0; rr < nr; ++rr) {
            const size_t off = (size_t)rp[r0 + rr] * N + rq[r0 + rr];
            double* dst = buf.data() + (size_t)rr * ld;
            for (int g = 0; g < f->n_chol; ++g) dst[g] = L[(size_t)g * N * N + off];
        }
        CK(cudaMemcpy(ops.dLt + (size_t)r0 * ld, buf.data(), (size_t)nr * ld * 8, cudaMemcpyHostToDevice));
    }
    return make_tmap(&ops.tmLt, ops.dLt, ld, (unsigned long long)ops.tri_pad, CO_BM);
}

// frees every device array of a multi-determinant plan and the plan itself
void free_cas_plan(CasPlan* c) {
    if (!c) return;
    void* cp[] = {c->dHoles, c->dParts, c->dCoef, c->dTh0, c->dA0, c->dT, c->dG, c->dWd, c->dEv, c->dSt0, c->dHoleIdx, c->dKind, c->dS, c->dH, c->dPart,
                  c->dStV, c->dHolesB, c->dPartsB, c->dTh0B, c->dA0B, c->dTB, c->dGB, c->dWdB, c->dSt0B, c->dHoleIdxB, c->dKindB, c->dSB, c->dHB,
                  c->dPartB, c->dStVB, c->dThAct[0], c->dThAct[1], c->dZ[0], c->dZ[1], c->dEJu, c->dPairs[0], c->dPairs[1], c->dPassAct[0], c->dPassAct[1]};
    for (void* q : cp)
        if (q) cudaFree(q);
    delete c;
}

void free_all(lo_factors* f) {
    if (!f) return;
    if (f->device >= 0) {
        cudaSetDevice(f->device);
        for (auto& ev : f->events) { cudaEventDestroy(ev.e0); cudaEventDestroy(ev.e1); }
        for (auto& ev : f->pool) { cudaEventDestroy(ev.e0); cudaEventDestroy(ev.e1); }
        f->bU.release();
        f->bW.release();
        free_cas_plan(f->cas);
        f->cas = nullptr;
        free_exchange_i8(f);
        if (f->copyStream) cudaStreamDestroy(f->copyStream);
        for (int c = 0; c < LO_HOST_CHUNKS; ++c)
            if (f->evCopy[c]) cudaEventDestroy(f->evCopy[c]);
        if (f->evEnter) cudaEventDestroy(f->evEnter);
        void* ptrs[] = {f->dSchedOff, f->dSchedTile, f->dWgt, f->dTiles, f->dTiles4, f->dEJLpart, f->dThT, f->dA[0], f->dA[1], f->dXpart, f->dEJpart, f->dEKpart,
                        f->dStatus, f->dEout, f->dStatusOut, f->dPhi[0], f->dPhi[1], f->dXT, f->dB};
        for (void* p : ptrs)
            if (p) cudaFree(p);
    }
    delete f;
}

// fetch packed rows [row0,row0+r) of U or W to a host buffer with pitch N
lo_status fetch_rows(const lo_factors* f, bool isU, long long row0, int r, double* dst) {
    if (r <= 0) return LO_OK;
    if (f->device >= 0) {
        CK(cudaSetDevice(f->device));
        const double* src = (isU ? f->dU : f->dW) + (size_t)row0 * f->N_pad;
        CK(cudaMemcpy2D(dst, (size_t)f->N * 8, src, (size_t)f->N_pad * 8, (size_t)f->N * 8, (size_t)r, cudaMemcpyDeviceToHost));
    } else {
        const std::vector<double>& v = isU ? f->hU : f->hW;
        for (int K = 0; K < r; ++K) std::memcpy(dst + (size_t)K * f->N, &v[(size_t)(row0 + K) * f->N_pad], (size_t)f->N * 8);
    }
    return LO_OK;
}

}  // namespace
}  // namespace lo

using namespace lo;

extern "C" {

const char* lo_last_error(void) { return err_buf().c_str(); }
const char* lo_version(void) { return "lo_afqmc_b200 0.1 (sm_100a)"; }

lo_status lo_setup(int N, int n_chol, int n_spin, const int n_occ[2], const double* h, const double* L, const double* psi_a,
                   const double* psi_b, double threshold, int device, int max_walkers, unsigned flags, lo_factors** out) {
    if (!out) { set_error("lo_setup: out is NULL"); return LO_EINVAL; }
    *out = nullptr;
    if (N <= 0 || n_chol <= 0 || (n_spin != 1 && n_spin != 2) || !n_occ || !h || !L || !psi_a || (n_spin == 2 && !psi_b) ||
        !(threshold >= 0.0) || max_walkers <= 0) {
        set_error("lo_setup: invalid argument (shape, NULL pointer, negative threshold or max_walkers <= 0)");
        return LO_EINVAL;
    }
    for (int s = 0; s < n_spin; ++s)
        if (n_occ[s] <= 0 || n_occ[s] > N) { set_error("lo_setup: n_occ out of range"); return LO_EINVAL; }
    int rsvd_k = 0;
    if (flags & LO_SETUP_RANDOMIZED_SVD) {
        // sketch size: bits 8..15 of flags in units of 16 rows, default 64; the sketches live in the V scratch of a block
        rsvd_k = (int)((flags >> 8) & 0xffu) * 16;
        if (rsvd_k == 0) rsvd_k = 64;
        if (rsvd_k > 128 || 4 * rsvd_k > N) rsvd_k = 0;       // block too small for a sketch to pay: full method only
    }
    if ((flags & (LO_SETUP_GPU_SVD | LO_SETUP_PROPAGATOR)) && device < 0) {
        set_error("lo_setup: LO_SETUP_GPU_SVD / LO_SETUP_PROPAGATOR need device >= 0");
        return LO_EINVAL;
    }

    const double t_enter = omp_get_wtime();
    lo_factors* f = new (std::nothrow) lo_factors();
    if (!f) { set_error("lo_setup: out of host memory"); return LO_ENOMEM; }
    f->N = N; f->N_pad = round_up(N, KTILE); f->n_chol = n_chol; f->Xp = round_up(n_chol + 1, CO_BM);
    f->n_spin = n_spin; f->threshold = threshold; f->device = device; f->max_walkers = max_walkers;
    f->Wcap = round_up(max_walkers, WALKER_TILE); f->ldw = 2 * f->Wcap;
    for (int s = 0; s < n_spin; ++s) { f->n_occ[s] = n_occ[s]; f->o_base[s] = f->O_tot; f->O_tot += n_occ[s]; }
    f->ops = std::make_shared<SharedOps>();
    f->ops->device = device;
    const double* psi[2] = {psi_a, psi_b};
    lo_status st = LO_OK;
    try {
        if (device >= 0) {
            cudaError_t e = cudaSetDevice(device);
            if (e != cudaSuccess) { set_error(std::string("cudaSetDevice: ") + cudaGetErrorString(e)); free_all(f); return LO_ECUDA; }
            cudaDeviceProp prop;
            cudaGetDeviceProperties(&prop, device);
            f->num_sms = prop.multiProcessorCount;
            for (int s = 0; s < n_spin; ++s) {
                size_t b = (size_t)N * n_occ[s] * 8;
                if (cudaMalloc(&f->ops->dPsi[s], b) != cudaSuccess || cudaMemcpy(f->ops->dPsi[s], psi[s], b, cudaMemcpyHostToDevice) != cudaSuccess) {
                    set_error("lo_setup: cannot upload psi"); free_all(f); return LO_ECUDA;
                }
            }
        }
        // ---- half rotation (always kept on the host as well: lo_retruncate / accessors / host-only sets)
        host_half_rotate(N, n_chol, n_spin, f->n_occ, f->o_base, f->O_tot, h, L, psi, f->ops->hLbar);
        if (device >= 0) {
            st = upload_lbar(f);
            if (st == LO_OK && (flags & LO_SETUP_PROPAGATOR)) st = upload_lt(f, L);
            if (st != LO_OK) { free_all(f); return st; }
        }
        // ---- rigorous pre-SVD pair screen: Y^{ij} = sum_g l^g_i (l^g_j)^T with l^g_i = Lbar[g][i][:],
        // so sigma_1(Y^{ij}) <= |Y^{ij}|_F <= sum_g |l^g_i|_2 |l^g_j|_2.  A pair whose bound is <= threshold has rank 0 under
        // Eq. 18 whatever its SVD says: neither its block nor its SVD is formed.  (The bound keeps the locality of every
        // Cholesky vector, so it decays with the distance between the two orbitals.)
        const bool prescreen = !(flags & LO_SETUP_NO_PRESCREEN);
        std::vector<double> lnorm((size_t)n_chol * f->O_tot);
        {
            const double* Lb = f->ops->hLbar.data();
#pragma omp parallel for schedule(static)
            for (long long go = 0; go < (long long)n_chol * f->O_tot; ++go) {
                const double* v = Lb + (size_t)go * N;
                double a = 0;
                for (int p = 0; p < N; ++p) a += v[p] * v[p];
                lnorm[go] = std::sqrt(a);
            }
        }
        auto pair_bound = [&](int oi, int oj) {
            double b = 0;
            for (int g = 0; g < n_chol; ++g) b += lnorm[(size_t)g * f->O_tot + oi] * lnorm[(size_t)g * f->O_tot + oj];
            return b * (1.0 + 1e-12);       // rounding of the sum itself
        };
        // ---- per-pair SVD + truncation + packing, batch by batch in layout order (whole L2 blocks per batch)
        std::vector<PairRec> pairs;
        std::vector<size_t> bstart;
        enumerate_blocks(f, pairs, bstart);
        st = begin_pack(f);
        if (st != LO_OK) { free_all(f); return st; }
        const bool on_gpu = (flags & LO_SETUP_GPU_SVD) != 0;
        f->setup_on_gpu = on_gpu ? 1 : 0;
        f->rsvd_k = rsvd_k;
        size_t B = 256;   // pairs per batch
        double *tY = nullptr, *tV = nullptr, *tU = nullptr, *tW = nullptr, *dSig = nullptr;
        int* dOrd = nullptr;
        auto free_tmp = [&]() { cudaFree(tY); cudaFree(tV); cudaFree(tU); cudaFree(tW); cudaFree(dSig); cudaFree(dOrd); };
        if (on_gpu) {
            const size_t per_pair = gpu_pair_svd_bytes_per_pair(N, f->N_pad);
            size_t free_b = 0, total_b = 0;
            cudaMemGetInfo(&free_b, &total_b);
            B = std::max<size_t>(1, std::min<size_t>({pairs.size(), (size_t)(f->num_sms * 4), (free_b / 8) / per_pair}));
            const size_t mat = (size_t)N * f->N_pad * 8;
            if (cudaMalloc(&tY, B * mat) != cudaSuccess || cudaMalloc(&tV, B * mat) != cudaSuccess || cudaMalloc(&tU, B * mat) != cudaSuccess ||
                cudaMalloc(&tW, B * mat) != cudaSuccess || cudaMalloc(&dSig, B * N * 8) != cudaSuccess || cudaMalloc(&dOrd, B * N * 4) != cudaSuccess) {
                set_error("lo_setup: cannot allocate GPU SVD workspace"); free_tmp(); free_all(f); return LO_ENOMEM;
            }
        }
        std::vector<double> hSig(B * N);
        std::vector<std::vector<double>> pU(on_gpu ? 0 : B), pW(on_gpu ? 0 : B);
        std::vector<int> bi(B), bj(B);
        std::vector<GatherRec> table;
        const double* Lbar = f->ops->hLbar.data();
        for (size_t blk = 0; blk + 1 < bstart.size() && st == LO_OK;) {
            // batch = consecutive whole blocks of one spin, at most B pairs (a block larger than B is split)
            const size_t k0 = bstart[blk];
            const int spin = pairs[k0].spin;
            size_t k1 = k0, blk1 = blk;
            while (blk1 + 1 < bstart.size() && pairs[bstart[blk1]].spin == spin && bstart[blk1 + 1] - k0 <= B) k1 = bstart[++blk1];
            const bool split = (k1 == k0);
            if (split) k1 = std::min(k0 + B, bstart[blk + 1]);
            const int n_all = (int)(k1 - k0);
            int n = 0;                       // pairs of the batch that survive the pre-SVD screen: slots 0..n-1 of the SVD batch
            for (int y = 0; y < n_all; ++y) {
                PairRec& pr = pairs[k0 + y];
                const double bound = prescreen ? pair_bound(f->o_base[spin] + pr.i, f->o_base[spin] + pr.j) : 0.0;
                if (prescreen && bound <= threshold) { pr.x = -1; pr.r = 0; pr.snext = bound; ++f->n_prescreened; continue; }
                pr.x = n; bi[n] = pr.i; bj[n] = pr.j; ++n;
            }
            std::vector<SvdStat> stats_of_batch;
            const double t_svd = omp_get_wtime();
            const double skip_below = prescreen ? threshold : -1.0;     // second screen: |Y|_F <= threshold, known once Y is formed
            if (n == 0) {
            } else if (on_gpu) {
                st = rsvd_k ? gpu_pair_rsvd(f, spin, bi.data(), bj.data(), n, rsvd_k, tY, tV, tU, tW, dSig, dOrd, hSig.data(), skip_below, &f->svd_stat,
                                            &f->n_rsvd_accepted)
                            : gpu_pair_svd(f, spin, bi.data(), bj.data(), n, tY, tV, tU, tW, dSig, dOrd, hSig.data(), skip_below, &f->svd_stat);
                if (st != LO_OK) break;
            } else {
                stats_of_batch.assign(n, SvdStat());
                std::vector<SvdStat>& stats = stats_of_batch;
                int oom = 0;       // an allocation failure inside the parallel region must not escape it
#pragma omp parallel
                {
                    std::vector<double> G, V, sg, rU, rW;
                    std::vector<int> order;
                    try { G.resize((size_t)N * N); V.resize((size_t)N * N); } catch (const std::bad_alloc&) {
#pragma omp atomic write
                        oom = 1;
                    }
#pragma omp for schedule(dynamic, 1)
                    for (int x = 0; x < n; ++x) {
                        if (G.size() != (size_t)N * N || V.size() != (size_t)N * N) continue;
                        try {
                        host_pair_gram_t(N, n_chol, f->O_tot, Lbar, f->o_base[spin] + bi[x], f->o_base[spin] + bj[x], G.data());
                        if (rsvd_k && host_pair_rsvd(N, rsvd_k, G.data(), sg, rU, rW, &stats[x])) {
                            // the sketch captured the block: its factors are the SVD to working accuracy
                            sg.resize(N, 0.0);
                            std::copy(sg.begin(), sg.end(), hSig.begin() + (size_t)x * N);
                            int r = 0;
                            while (r < rsvd_k && sg[r] > threshold) ++r;
                            pU[x].assign(rU.begin(), rU.begin() + (size_t)r * N);
                            pW[x].assign(rW.begin(), rW.begin() + (size_t)r * N);
#pragma omp atomic
                            ++f->n_rsvd_accepted;
                            continue;
                        }
                        host_block_svd(N, N, G.data(), V.data(), sg, order, skip_below, &stats[x]);
                        std::copy(sg.begin(), sg.end(), hSig.begin() + (size_t)x * N);
                        int r = 0;
                        while (r < N && sg[r] > threshold) ++r;
                        pU[x].resize((size_t)r * N);
                        pW[x].resize((size_t)r * N);
                        for (int K = 0; K < r; ++K) {
                            const double* g = &G[(size_t)order[K] * N];
                            const double inv = 1.0 / sg[K];
                            for (int e = 0; e < N; ++e) pU[x][(size_t)K * N + e] = g[e] * inv;
                            std::memcpy(&pW[x][(size_t)K * N], &V[(size_t)order[K] * N], (size_t)N * 8);
                        }
                        } catch (const std::bad_alloc&) {
#pragma omp atomic write
                            oom = 1;
                        }
                    }
                }
                if (oom) { set_error("lo_setup: out of host memory in the pair SVDs"); st = LO_ENOMEM; break; }
            }
            f->setup_svd_seconds += omp_get_wtime() - t_svd;
            if (!on_gpu)
                for (const SvdStat& t : stats_of_batch) {
                    f->svd_stat.sweeps = std::max(f->svd_stat.sweeps, t.sweeps);
                    f->svd_stat.offdiag = std::max(f->svd_stat.offdiag, t.offdiag);
                    if (!t.converged) f->svd_stat.converged = false;
                    f->svd_stat.screened += t.screened;
                }
            if (!f->svd_stat.converged) {
                set_error("lo_setup: the pair-block SVD did not converge within " + std::to_string(SVD_MAX_SWEEPS) + " sweeps (largest remaining "
                          "normalised off-diagonal " + std::to_string(f->svd_stat.offdiag) + ")");
                st = LO_EINTERNAL;
                break;
            }
            for (int y = 0; y < n_all; ++y) {
                PairRec& pr = pairs[k0 + y];
                if (pr.x < 0) continue;
                const double* sg = &hSig[(size_t)pr.x * N];
                int r = 0;
                while (r < N && sg[r] > threshold) ++r;
                pr.r = r;
                pr.snext = r < N ? sg[r] : 0.0;
            }
            table.clear();
            auto sig = [&](const PairRec& pr, int K) { return hSig[(size_t)pr.x * N + K]; };
            auto src = [&](const PairRec& pr) { return (long long)pr.x * N; };
            if (split) layout_block(f, &pairs[k0], &pairs[k0] + n_all, sig, src, table);
            else
                for (size_t bb = blk; bb < blk1; ++bb) layout_block(f, &pairs[bstart[bb]], &pairs[bstart[bb + 1]], sig, src, table);
            st = grow_pack(f);
            if (st != LO_OK) break;
            if (on_gpu) {
                st = gpu_gather_rows(tU, f->dU, table.data(), (int)table.size(), f->N_pad);
                if (st == LO_OK) st = gpu_gather_rows(tW, f->dW, table.data(), (int)table.size(), f->N_pad);
            } else {
                for (const GatherRec& g : table) {
                    const int x = (int)(g.src_row / N);
                    if (device >= 0) {
                        if (cudaMemcpy2D(f->dU + (size_t)g.dst_row * f->N_pad, (size_t)f->N_pad * 8, pU[x].data(), (size_t)N * 8, (size_t)N * 8, g.r, cudaMemcpyHostToDevice) != cudaSuccess ||
                            cudaMemcpy2D(f->dW + (size_t)g.dst_row * f->N_pad, (size_t)f->N_pad * 8, pW[x].data(), (size_t)N * 8, (size_t)N * 8, g.r, cudaMemcpyHostToDevice) != cudaSuccess) {
                            set_error("lo_setup: factor upload failed"); st = LO_ECUDA; break;
                        }
                    } else {
                        for (int K = 0; K < g.r; ++K) {
                            std::memcpy(&f->hU[(size_t)(g.dst_row + K) * f->N_pad], &pU[x][(size_t)K * N], (size_t)N * 8);
                            std::memcpy(&f->hW[(size_t)(g.dst_row + K) * f->N_pad], &pW[x][(size_t)K * N], (size_t)N * 8);
                        }
                    }
                }
            }
            if (split && k1 < bstart[blk + 1]) { bstart[blk] = k1; }   // rest of the oversized block next time
            else blk = split ? blk + 1 : blk1;
        }
        if (on_gpu) free_tmp();
        if (st == LO_OK) st = finish_pack(f);
        if (st != LO_OK) { free_all(f); return st; }
    } catch (const std::bad_alloc&) {
        set_error("lo_setup: out of host memory");
        free_all(f);
        return LO_ENOMEM;
    }
    f->setup_seconds = omp_get_wtime() - t_enter;
    *out = f;
    return LO_OK;
}

lo_status lo_info_get(const lo_factors* f, lo_info* info) {
    if (!f || !info) { set_error("lo_info_get: NULL argument"); return LO_EINVAL; }
    std::memset(info, 0, sizeof(*info));
    info->N = f->N; info->n_chol = f->n_chol; info->n_spin = f->n_spin; info->N_pad = f->N_pad;
    int mx = 0, mn = f->N;
    for (int s = 0; s < f->n_spin; ++s) {
        info->n_occ[s] = f->n_occ[s];
        info->n_pairs[s] = (long long)f->rank[s].size();
        long long sum = 0;
        for (int r : f->rank[s]) { sum += r; mx = std::max(mx, r); mn = std::min(mn, r); }
        info->sum_rank[s] = sum;
    }
    info->sum_rank_padded = f->rows; info->max_rank = mx; info->min_rank = mn;
    info->factor_bytes = f->factor_bytes; info->lbar_bytes = f->lbar_bytes; info->workspace_bytes = f->workspace_bytes;
    info->threshold = f->threshold; info->device = f->device; info->max_walkers = f->max_walkers;
    info->setup_on_gpu = f->setup_on_gpu; info->n_tiles = f->n_tiles;
    info->svd_sweeps_max = f->svd_stat.sweeps; info->svd_offdiag_max = f->svd_stat.offdiag;
    info->setup_seconds = f->setup_seconds; info->setup_svd_seconds = f->setup_svd_seconds;
    info->rsvd_sketch = f->rsvd_k; info->n_pairs_rsvd = f->n_rsvd_accepted;
    info->n_pairs_prescreened = f->n_prescreened + f->svd_stat.screened;
    info->n_pairs_energy_screened = f->n_energy_screened; info->energy_screen_cutoff = f->energy_cutoff;
    info->energy_screen_bound = f->energy_bound;
    info->exchange_mode = f->ex_mode;
    info->int8_bytes = f->i8_bytes;
    return LO_OK;
}

lo_status lo_ranks(const lo_factors* f, int spin, int* r) {
    if (!f || !r || spin < 0 || spin >= f->n_spin) { set_error("lo_ranks: invalid argument"); return LO_EINVAL; }
    std::copy(f->rank[spin].begin(), f->rank[spin].end(), r);
    return LO_OK;
}

lo_status lo_factor_pair(const lo_factors* f, int spin, int i, int j, double* U, double* sigma, double* W) {
    if (!f || spin < 0 || spin >= f->n_spin || i < 0 || j < i || j >= f->n_occ[spin]) { set_error("lo_factor_pair: invalid argument"); return LO_EINVAL; }
    const int O = f->n_occ[spin];
    const size_t k = (size_t)i * O - (size_t)i * (i - 1) / 2 + (j - i);
    const int r = f->rank[spin][k];
    const long long row0 = f->row_off[spin][k];
    lo_status st;
    if (U && (st = fetch_rows(f, true, row0, r, U)) != LO_OK) return st;
    if (W && (st = fetch_rows(f, false, row0, r, W)) != LO_OK) return st;
    if (sigma && r > 0) {
        const double scale = -(f->n_spin == 1 ? 1.0 : 0.5) * (i == j ? 1.0 : 2.0);   // power of two: exact
        for (int K = 0; K < r; ++K) sigma[K] = f->hWgt[(size_t)row0 + K] / scale;
    }
    return LO_OK;
}

lo_status lo_factor_all(const lo_factors* f, int spin, double* U, double* sigma, double* W) {
    if (!f || spin < 0 || spin >= f->n_spin) { set_error("lo_factor_all: invalid argument"); return LO_EINVAL; }
    const int O = f->n_occ[spin];
    size_t off = 0, k = 0;
    for (int i = 0; i < O; ++i)
        for (int j = i; j < O; ++j, ++k) {
            lo_status st = lo_factor_pair(f, spin, i, j, U ? U + off * f->N : nullptr, sigma ? sigma + off : nullptr, W ? W + off * f->N : nullptr);
            if (st != LO_OK) return st;
            off += f->rank[spin][k];
        }
    return LO_OK;
}

// New factor set from the rows of `f`: every pair keeps the prefix sigma_K > looser of its rows (lo_retruncate), and a
// pair with m_ij sigma_1 <= pair_cutoff keeps none (lo_screen_pairs).
static lo_status rebuild_from(const lo_factors* f, double looser, double pair_cutoff, lo_factors** out) {
    *out = nullptr;
    lo_factors* g = new (std::nothrow) lo_factors();
    if (!g) { set_error("lo_retruncate / lo_screen_pairs: out of host memory"); return LO_ENOMEM; }
    g->N = f->N; g->N_pad = f->N_pad; g->n_chol = f->n_chol; g->Xp = f->Xp; g->n_spin = f->n_spin; g->O_tot = f->O_tot;
    for (int s = 0; s < 2; ++s) { g->n_occ[s] = f->n_occ[s]; g->o_base[s] = f->o_base[s]; }
    g->threshold = looser; g->device = f->device; g->max_walkers = f->max_walkers; g->Wcap = f->Wcap; g->ldw = f->ldw;
    g->num_sms = f->num_sms; g->setup_on_gpu = f->setup_on_gpu; g->svd_stat = f->svd_stat; g->ops = f->ops; g->lbar_bytes = f->lbar_bytes;
    g->rsvd_k = f->rsvd_k; g->n_rsvd_accepted = f->n_rsvd_accepted;
    g->n_prescreened = f->n_prescreened; g->setup_seconds = f->setup_seconds; g->setup_svd_seconds = f->setup_svd_seconds;
    g->n_energy_screened = f->n_energy_screened; g->energy_cutoff = std::max(f->energy_cutoff, pair_cutoff); g->energy_bound = f->energy_bound;
    try {
        std::vector<PairRec> pairs;
        std::vector<size_t> bstart;
        enumerate_blocks(g, pairs, bstart);
        lo_status st = begin_pack(g);
        if (st != LO_OK) { free_all(g); return st; }
        auto sigma_of = [&](const PairRec& pr, int K) {
            const double scale = -(f->n_spin == 1 ? 1.0 : 0.5) * (pr.i == pr.j ? 1.0 : 2.0);
            return f->hWgt[(size_t)pr.src + K] / scale;
        };
        for (PairRec& pr : pairs) {
            const size_t k = pair_index(f->n_occ[pr.spin], pr.i, pr.j);
            const int r0 = f->rank[pr.spin][k];
            pr.src = f->row_off[pr.spin][k];
            int r = 0;
            while (r < r0 && sigma_of(pr, r) > looser) ++r;
            if (r > 0 && pair_cutoff > 0.0) {
                // energy screen: |m_ij sum_K sigma_K a_K b_K| <= m_ij sigma_1 |Theta_i||Theta_j|
                const double ms1 = (pr.i == pr.j ? 1.0 : 2.0) * sigma_of(pr, 0);
                if (ms1 <= pair_cutoff) {
                    r = 0;
                    ++g->n_energy_screened;
                    g->energy_bound += (f->n_spin == 1 ? 1.0 : 0.5) * ms1;
                }
            }
            pr.r = r;
            pr.snext = r < r0 ? sigma_of(pr, r) : f->sigma_next[pr.spin][k];
        }
        std::vector<GatherRec> table;
        auto src = [&](const PairRec& pr) { return pr.src; };
        for (size_t blk = 0; blk + 1 < bstart.size(); ++blk) layout_block(g, &pairs[bstart[blk]], &pairs[bstart[blk + 1]], sigma_of, src, table);
        st = grow_pack(g);
        if (st == LO_OK) {
            if (g->device >= 0) {
                st = gpu_gather_rows(f->dU, g->dU, table.data(), (int)table.size(), g->N_pad);
                if (st == LO_OK) st = gpu_gather_rows(f->dW, g->dW, table.data(), (int)table.size(), g->N_pad);
            } else {
                for (const GatherRec& t : table) {
                    std::memcpy(&g->hU[(size_t)t.dst_row * g->N_pad], &f->hU[(size_t)t.src_row * g->N_pad], (size_t)t.r * g->N_pad * 8);
                    std::memcpy(&g->hW[(size_t)t.dst_row * g->N_pad], &f->hW[(size_t)t.src_row * g->N_pad], (size_t)t.r * g->N_pad * 8);
                }
            }
        }
        if (st == LO_OK) st = finish_pack(g);
        if (st != LO_OK) { free_all(g); return st; }
    } catch (const std::bad_alloc&) {
        set_error("lo_retruncate / lo_screen_pairs: out of host memory");
        free_all(g);
        return LO_ENOMEM;
    }
    *out = g;
    return LO_OK;
}

lo_status lo_retruncate(const lo_factors* f, double looser, lo_factors** out) {
    if (!f || !out || !(looser >= f->threshold)) { set_error("lo_retruncate: invalid argument (threshold must be >= the original)"); return LO_EINVAL; }
    return rebuild_from(f, looser, 0.0, out);
}

lo_status lo_screen_pairs(const lo_factors* f, double pair_cutoff, lo_factors** out) {
    if (!f || !out || !(pair_cutoff >= 0.0)) { set_error("lo_screen_pairs: invalid argument (cutoff must be >= 0)"); return LO_EINVAL; }
    return rebuild_from(f, f->threshold, pair_cutoff, out);
}

static lo_status check_call(const lo_factors* f, int n_w, const void* phi_a, const void* phi_b) {
    if (!f) { set_error("lo_local_energy: factors is NULL"); return LO_EINVAL; }
    if (f->device < 0) { set_error("lo_local_energy: factor set was built without a device (device < 0); there is no CPU path"); return LO_ECUDA; }
    if (n_w <= 0 || n_w > f->max_walkers) { set_error("lo_local_energy: n_w out of range (1..max_walkers)"); return LO_EINVAL; }
    if (n_w > 65535) { set_error("lo_local_energy: at most 65535 walkers per call (grid dimension of the S1 kernels); split the batch"); return LO_EINVAL; }
    if (!phi_a || (f->n_spin == 2 && !phi_b)) { set_error("lo_local_energy: phi is NULL"); return LO_EINVAL; }
    if (((uintptr_t)phi_a & 15) || ((uintptr_t)phi_b & 15)) { set_error("lo_local_energy: phi must be 16-byte aligned"); return LO_EINVAL; }
    return LO_OK;
}

lo_status lo_local_energy(const lo_factors* fc, int n_w, const void* phi_a, const void* phi_b, void* E_L, void* E1, void* E_J, void* E_K,
                          int* walker_status, void* stream) {
    lo_status st = check_call(fc, n_w, phi_a, phi_b);
    if (st != LO_OK) return st;
    if (!E_L) { set_error("lo_local_energy: E_L is NULL"); return LO_EINVAL; }
    if (((uintptr_t)E_L & 15) || ((uintptr_t)E1 & 15) || ((uintptr_t)E_J & 15) || ((uintptr_t)E_K & 15)) {
        set_error("lo_local_energy: outputs must be 16-byte aligned");
        return LO_EINVAL;
    }
    lo_factors* f = const_cast<lo_factors*>(fc);
    CK(cudaSetDevice(f->device));
    return launch_local_energy(f, n_w, phi_a, phi_b, E_L, E1, E_J, E_K, walker_status, nullptr, (cudaStream_t)stream);
}

lo_status lo_local_energy_host(const lo_factors* fc, int n_w, const void* phi_a_host, const void* phi_b_host, void* E_host, int* status_host,
                               void* stream) {
    lo_status st = check_call(fc, n_w, phi_a_host, phi_b_host);
    if (st != LO_OK) return st;
    if (!E_host) { set_error("lo_local_energy_host: E_host is NULL"); return LO_EINVAL; }
    lo_factors* f = const_cast<lo_factors*>(fc);
    cudaStream_t s = (cudaStream_t)stream;
    CK(cudaSetDevice(f->device));
    // Walker chunks (starting at multiples of 64, at most LO_HOST_CHUNKS): the H2D copy of chunk c+1 runs on
    // a private copy stream while the kernels of chunk c run on `s`; walkers are independent, so a chunk is a complete
    // pass of the hot path over its walkers (the factor rows are streamed once per chunk).
    const char* ph[2] = {static_cast<const char*>(phi_a_host), static_cast<const char*>(phi_b_host)};
    // Chunk sizes grow geometrically (64, 128, 256, rest): the first copy -- the only one nothing can hide -- is short, and
    // every later chunk's copy is no longer than the kernels of the chunk before it even in the small-rank regime (a walker
    // costs about twice as long to process as to copy there), while most walkers still run in one large, efficient launch.
    int chunk[LO_HOST_CHUNKS], n_chunks = 0;
    {
        int rem = n_w, c = WALKER_TILE;
        if (n_w >= 4 * WALKER_TILE)
            while (n_chunks < LO_HOST_CHUNKS - 1 && rem > 3 * c) { chunk[n_chunks++] = c; rem -= c; c *= 2; }
        chunk[n_chunks++] = rem;
    }
    // The copies are ordered after everything already queued on the caller's stream (a stream-ordered producer of the
    // pinned Phi buffer, or an earlier call on this handle that still reads the staging area).
    CK(cudaEventRecord(f->evEnter, s));
    CK(cudaStreamWaitEvent(f->copyStream, f->evEnter, 0));
    auto body = [&]() -> lo_status {
        for (int c = 0, w0 = 0; c < n_chunks; w0 += chunk[c], ++c) {
            const int nc = chunk[c];
            for (int sp = 0; sp < f->n_spin; ++sp) {
                const size_t per_w = (size_t)f->N * f->n_occ[sp] * 16;
                CK(cudaMemcpyAsync(reinterpret_cast<char*>(f->dPhi[sp]) + w0 * per_w, ph[sp] + w0 * per_w, nc * per_w, cudaMemcpyHostToDevice, f->copyStream));
            }
            CK(cudaEventRecord(f->evCopy[c], f->copyStream));
        }
        for (int c = 0, w0 = 0; c < n_chunks; w0 += chunk[c], ++c) {
            const int nc = chunk[c];
            CK(cudaStreamWaitEvent(s, f->evCopy[c], 0));
            const char* pa = reinterpret_cast<const char*>(f->dPhi[0]) + (size_t)w0 * f->N * f->n_occ[0] * 16;
            const char* pb = f->n_spin == 2 ? reinterpret_cast<const char*>(f->dPhi[1]) + (size_t)w0 * f->N * f->n_occ[1] * 16 : nullptr;
            lo_status st2 = launch_local_energy(f, nc, pa, pb, nullptr, nullptr, nullptr, nullptr, f->dStatusOut + w0, f->dEout + (size_t)w0 * 8, s);
            if (st2 != LO_OK) return st2;
        }
        CK(cudaMemcpyAsync(E_host, f->dEout, (size_t)n_w * 4 * 16, cudaMemcpyDeviceToHost, s));
        if (status_host) CK(cudaMemcpyAsync(status_host, f->dStatusOut, (size_t)n_w * 4, cudaMemcpyDeviceToHost, s));
        return LO_OK;
    };
    st = body();
    // success or not, nothing of this call is left in flight when it returns (the host buffers are the caller's)
    const cudaError_t e1 = cudaStreamSynchronize(f->copyStream), e2 = cudaStreamSynchronize(s);
    if (st == LO_OK && (e1 != cudaSuccess || e2 != cudaSuccess)) {
        set_error(std::string("lo_local_energy_host: ") + cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
        st = LO_ECUDA;
    }
    return st;
}

lo_status lo_coulomb_x(const lo_factors* f, const void** X_dev, int* ld) {
    if (!f || !X_dev || !ld) { set_error("lo_coulomb_x: NULL argument"); return LO_EINVAL; }
    if (f->device < 0) { set_error("lo_coulomb_x: no device"); return LO_ECUDA; }
    *X_dev = f->dXpart;
    *ld = f->Wcap;
    return LO_OK;
}

lo_status lo_set_coulomb_mode(lo_factors* f, int mode) {
    if (!f || (mode != LO_COULOMB_CHOLESKY && mode != LO_COULOMB_COMPRESSED)) { set_error("lo_set_coulomb_mode: invalid argument"); return LO_EINVAL; }
    if (mode == LO_COULOMB_COMPRESSED && f->n_spin != 1) {
        set_error("lo_set_coulomb_mode: the compressed Coulomb term needs opposite-spin pair blocks, which an unrestricted factor set does not hold");
        return LO_EINVAL;
    }
    f->coulomb_lo = mode == LO_COULOMB_COMPRESSED ? 1 : 0;
    return LO_OK;
}

lo_status lo_set_exchange_mode(lo_factors* f, int mode) {
    if (!f || (mode != LO_EXCHANGE_DMMA && mode != LO_EXCHANGE_INT8)) { set_error("lo_set_exchange_mode: invalid argument"); return LO_EINVAL; }
    if (mode == LO_EXCHANGE_INT8) {
        if (f->device < 0) { set_error("lo_set_exchange_mode: LO_EXCHANGE_INT8 needs a device-resident factor set"); return LO_EINVAL; }
        // exact int32 digit sums: 7 products of |digit| <= 64 per multiply-add, over N basis functions (exchange, Coulomb per orbital)
        // or n_chol fields (propagator): 7 * 4096 * K < 2^31
        if (f->N_pad > 65536 || (f->ops->dLt && f->ops->Xk_pad > 65536)) {
            set_error("lo_set_exchange_mode: LO_EXCHANGE_INT8 supports N (and n_chol with the propagator) up to 65536");
            return LO_EINVAL;
        }
        lo_status st = build_exchange_i8(f);      // slices the factor rows on first use
        if (st != LO_OK) return st;
    }
    f->ex_mode = mode;
    return LO_OK;
}

// validates one spin's excitation lists (shared by lo_set_cas_trial and lo_set_cas_trial_beta)
static lo_status check_strings(int n_det, int max_exc, int n_ref, int n_orb, const int* holes, const int* parts) {
    for (int d = 0; d < n_det; ++d) {
        bool ended = false;
        for (int k = 0; k < max_exc; ++k) {
            const int h = holes[(size_t)d * max_exc + k], p = parts[(size_t)d * max_exc + k];
            if (h < 0 || p < 0) { if (h >= 0 || p >= 0) { set_error("lo_set_cas_trial: hole/particle lists of different length"); return LO_EINVAL; } ended = true; continue; }
            if (ended || h >= n_ref || p < n_ref || p >= n_orb) { set_error("lo_set_cas_trial: hole must be < n_ref, particle in [n_ref, n_occ), -1 padding at the end"); return LO_EINVAL; }
            for (int l = 0; l < k; ++l)
                if (holes[(size_t)d * max_exc + l] == h || parts[(size_t)d * max_exc + l] == p) { set_error("lo_set_cas_trial: repeated hole or particle in one determinant"); return LO_EINVAL; }
        }
    }
    return LO_OK;
}

// SMW-energy data of one spin (0: alpha / closed shell -> the plain fields of the plan, 1: beta -> the *B fields): hole
// indices into the active set, per-determinant orbital kinds, the S / H intermediates, partial sums, the Theta0 tensor map.
static lo_status alloc_smw_spin(lo_factors* f, CasPlan* c, int spin, const int* holes, const int* parts, const std::vector<int>& act) {
    const int n_orb = f->n_occ[spin], n_ref = spin == 0 ? c->n_ref : c->n_ref_b, n_det = c->n_det, max_exc = c->max_exc;
    const size_t nv = (size_t)c->max_real * n_det, ne = (size_t)n_det * max_exc;
    auto al = [&](void** p, size_t bytes) -> cudaError_t {
        cudaError_t e = cudaMalloc(p, std::max<size_t>(bytes, 16));
        if (e == cudaSuccess) e = cudaMemset(*p, 0, std::max<size_t>(bytes, 16));
        return e;
    };
    const int n_act = (int)act.size();
    const int na_pad = n_act <= 2 ? 2 : (n_act <= 4 ? 4 : 6);
    // up to 6 active columns: one pass on the panel list {x, y, A}; more: groups of 3 and one pass per pair of groups
    const int gs = n_act <= 6 ? 6 : 3, ng = n_act <= 6 ? 1 : (n_act + 2) / 3, npass = ng * (ng + 1) / 2;
    const int NP = ng == 1 ? 2 + na_pad : 8;
    std::vector<int> pass_act((size_t)npass * 6, 0);
    for (int a = 0, p = 0; a < ng; ++a)
        for (int b = a; b < ng; ++b, ++p)
            for (int l = 0; l < 6; ++l) {
                const int idx = ng == 1 ? l : (l < 3 ? a * 3 + l : b * 3 + (l - 3));
                pass_act[(size_t)p * 6 + l] = idx < n_act ? act[idx] : 0;
            }
    const int ce = std::max(1, std::min(16, (40 * 1024) / (npass * NP * NP * 16)));      // k_cas_energy keeps a chunk in <= 40 KB of shared memory
    // pairs of this spin that have rows, each with its range of <= 4-fragment tiles (consecutive in the tile list)
    std::vector<CasPair> hp;
    for (size_t t = 0; t < f->hTiles4.size(); ++t) {
        const ExTile& T = f->hTiles4[t];
        const bool mine = f->n_spin == 1 || (spin == 0 ? T.pi < f->o_base[1] : T.pi >= f->o_base[1]);
        if (!mine) continue;
        if (!hp.empty() && hp.back().pi == T.pi && hp.back().pj == T.pj && hp.back().t0 + hp.back().nt == (int)t) ++hp.back().nt;
        else hp.push_back({(int)t, 1, T.pi, T.pj});
    }
    const long long nt = (long long)hp.size();
    c->npair[spin] = nt;
    std::vector<int> hidx(ne + 16, -1);
    for (size_t k = 0; k < ne; ++k)
        if (holes[k] >= 0) hidx[k] = (int)(std::find(act.begin(), act.end(), holes[k]) - act.begin());
    for (int a = 0; a < 16; ++a) {
        hidx[ne + a] = a < n_act ? act[a] : 0;          // A_set (padded with column 0) behind the indices
        (spin == 0 ? c->hAct : c->hActB)[a] = hidx[ne + a];
    }
    std::vector<signed char> kind((size_t)n_det * n_orb);
    for (int d = 0; d < n_det; ++d)
        for (int x = 0; x < n_orb; ++x) {
            signed char kd = x < n_ref ? 0 : -1;
            for (int k = 0; k < max_exc; ++k) {
                if (holes[(size_t)d * max_exc + k] == x) kd = -1;
                if (parts[(size_t)d * max_exc + k] == x) kd = (signed char)(1 + k);
            }
            kind[(size_t)d * n_orb + x] = kd;
        }
    const int n_chunks = (int)((nt + ce - 1) / ce);
    c->gs[spin] = gs; c->ng[spin] = ng; c->npass[spin] = npass; c->ce[spin] = ce;
    int*& dHoleIdx = spin == 0 ? c->dHoleIdx : c->dHoleIdxB;
    signed char*& dKind = spin == 0 ? c->dKind : c->dKindB;
    int*& dStV = spin == 0 ? c->dStV : c->dStVB;
    double*& dS = spin == 0 ? c->dS : c->dSB;
    double*& dH = spin == 0 ? c->dH : c->dHB;
    double*& dPart = spin == 0 ? c->dPart : c->dPartB;
    double* dTh0 = spin == 0 ? c->dTh0 : c->dTh0B;
    (spin == 0 ? c->n_act : c->n_actB) = n_act;
    (spin == 0 ? c->NP : c->NPB) = NP;
    (spin == 0 ? c->n_chunks : c->n_chunksB) = n_chunks;
    CK(al((void**)&dHoleIdx, hidx.size() * 4));
    CK(al((void**)&dKind, kind.size()));
    CK(al((void**)&dStV, nv * 4));
    CK(al((void**)&dS, (size_t)npass * std::max<long long>(nt, 1) * c->max_real * NP * NP * 16));
    CK(al((void**)&dH, (size_t)c->W0cap * n_orb * CAS_HS * 16));
    CK(al((void**)&c->dPassAct[spin], pass_act.size() * 4));
    CK(cudaMemcpy(c->dPassAct[spin], pass_act.data(), pass_act.size() * 4, cudaMemcpyHostToDevice));
    CK(al((void**)&dPart, (size_t)std::max(n_chunks, 1) * nv * 2 * 16));
    CK(cudaMemcpy(dHoleIdx, hidx.data(), hidx.size() * 4, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(dKind, kind.data(), kind.size(), cudaMemcpyHostToDevice));
    CK(al((void**)&c->dPairs[spin], std::max<size_t>(hp.size(), 1) * sizeof(CasPair)));
    if (!hp.empty()) CK(cudaMemcpy(c->dPairs[spin], hp.data(), hp.size() * sizeof(CasPair), cudaMemcpyHostToDevice));
    lo_status st = make_tmap(spin == 0 ? &c->tmTh0 : &c->tmTh0B, dTh0, f->N_pad, (unsigned long long)n_orb * 2 * c->W0cap, 32);
    if (st != LO_OK) return st;
    if (f->n_spin == 2) {
        // Cholesky-route Coulomb term of the unrestricted SMW energy: gathered active panels and the Z intermediates
        const size_t ldw0 = 2 * (size_t)c->W0cap, zcols = (size_t)f->Xp * f->O_tot;
        CK(al((void**)&c->dThAct[spin], (size_t)na_pad * ldw0 * f->N_pad * 8));
        CK(al((void**)&c->dZ[spin], (size_t)na_pad * ldw0 * zcols * 8));
        st = make_tmap(&c->tmThAct[spin], c->dThAct[spin], f->N_pad, (unsigned long long)na_pad * ldw0, 128);
        if (st == LO_OK && spin == 0) st = make_tmap(&c->tmLbarRows, f->ops->dLbar, f->N_pad, (unsigned long long)zcols, 128);
        if (st != LO_OK) return st;
        if (!c->dEJu) CK(al((void**)&c->dEJu, nv * 16));
    }
    return LO_OK;
}

// allocates and fills plan `c` (already sized); any failure leaves the partial allocations in `c` for the caller to free
static lo_status fill_cas_plan(lo_factors* f, CasPlan* c, const int* holes, const int* parts, const double* coef, const std::vector<int>& act) {
    const int n_orb = f->n_occ[0], n_ref = c->n_ref, n_det = c->n_det, max_exc = c->max_exc;
    const size_t nv = (size_t)c->max_real * n_det, ne = (size_t)n_det * max_exc;
    auto al = [&](void** p, size_t bytes) -> cudaError_t {
        cudaError_t e = cudaMalloc(p, std::max<size_t>(bytes, 16));
        if (e == cudaSuccess) e = cudaMemset(*p, 0, std::max<size_t>(bytes, 16));
        return e;
    };
    CK(al((void**)&c->dHoles, ne * 4));
    CK(al((void**)&c->dParts, ne * 4));
    CK(al((void**)&c->dCoef, (size_t)n_det * 8));
    CK(al((void**)&c->dTh0, (size_t)n_orb * 2 * c->W0cap * f->N_pad * 8));      // virtual panels stay zero
    CK(al((void**)&c->dA0, (size_t)c->W0cap * n_ref * n_ref * 16));
    CK(al((void**)&c->dT, (size_t)c->W0cap * std::max(c->n_virt, 1) * n_ref * 16));
    CK(al((void**)&c->dG, nv * max_exc * n_orb * 16));
    CK(al((void**)&c->dWd, nv * 16));
    CK(al((void**)&c->dEv, nv * 4 * 16));
    CK(al((void**)&c->dSt0, (size_t)c->W0cap * 4));
    CK(cudaMemcpy(c->dHoles, holes, ne * 4, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(c->dParts, parts, ne * 4, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(c->dCoef, coef, (size_t)n_det * 8, cudaMemcpyHostToDevice));
    if (c->mode == LO_CAS_SMW_ENERGY) {
        lo_status st = alloc_smw_spin(f, c, 0, holes, parts, act);
        if (st != LO_OK) return st;
    }
    return LO_OK;
}

lo_status lo_set_cas_trial(lo_factors* f, int n_ref, int n_det, int max_exc, const int* holes, const int* parts, const double* coef,
                           int max_real_walkers, int mode) {
    if (!f || !holes || !parts || !coef) { set_error("lo_set_cas_trial: NULL argument"); return LO_EINVAL; }
    if (f->device < 0) { set_error("lo_set_cas_trial: no device"); return LO_ECUDA; }
    const int n_orb = f->n_occ[0];
    if (mode != LO_CAS_DIRECT && mode != LO_CAS_SMW_ENERGY) { set_error("lo_set_cas_trial: mode must be LO_CAS_DIRECT or LO_CAS_SMW_ENERGY"); return LO_EINVAL; }
    if (n_ref <= 0 || n_ref > n_orb || n_det <= 0 || max_exc <= 0 || max_exc > CAS_MAX_EXC || max_real_walkers <= 0 ||
        (mode == LO_CAS_DIRECT && (long long)max_real_walkers * n_det > f->max_walkers) || max_real_walkers > f->max_walkers) {
        set_error("lo_set_cas_trial: invalid sizes (need 0 < n_ref <= n_occ, 1 <= max_exc <= 8, max_real_walkers * n_det <= max_walkers "
                  "in LO_CAS_DIRECT mode, max_real_walkers <= max_walkers)");
        return LO_EINVAL;
    }
    lo_status st = check_strings(n_det, max_exc, n_ref, n_orb, holes, parts);
    if (st != LO_OK) return st;
    // active set = the reference columns that are a hole in some determinant (the columns of A^-1 the SMW corrections touch)
    std::vector<int> act;
    for (size_t k = 0; k < (size_t)n_det * max_exc; ++k)
        if (holes[k] >= 0 && std::find(act.begin(), act.end(), holes[k]) == act.end()) act.push_back(holes[k]);
    std::sort(act.begin(), act.end());
    if (mode == LO_CAS_SMW_ENERGY && (int)act.size() > (f->n_spin == 1 ? CAS_MAX_ACT : 6)) {
        set_error("lo_set_cas_trial: LO_CAS_SMW_ENERGY supports at most 12 distinct hole columns (active occupied orbitals) for a closed-shell "
                  "trial and 6 per spin for an unrestricted one; use LO_CAS_DIRECT");
        return LO_EINVAL;
    }
    CK(cudaSetDevice(f->device));
    // The new plan is built aside and installed only when every allocation and upload has succeeded; on failure the
    // partial plan is freed and the previous trial (if any) stays in place.
    CasPlan* c = new (std::nothrow) CasPlan();
    if (!c) { set_error("lo_set_cas_trial: out of host memory"); return LO_ENOMEM; }
    c->n_ref = n_ref; c->n_det = n_det; c->max_exc = max_exc; c->n_virt = n_orb - n_ref; c->max_real = max_real_walkers;
    c->W0cap = round_up(max_real_walkers, WALKER_TILE);
    c->mode = mode;
    c->n_act = (int)act.size();
    st = fill_cas_plan(f, c, holes, parts, coef, act);
    if (st != LO_OK) {
        free_cas_plan(c);
        cudaGetLastError();      // an allocation failure is not sticky; clear it
        return st;
    }
    free_cas_plan(f->cas);
    f->cas = c;
    return LO_OK;
}

lo_status lo_set_cas_trial_beta(lo_factors* f, int n_ref_b, const int* holes_b, const int* parts_b) {
    if (!f || !holes_b || !parts_b) { set_error("lo_set_cas_trial_beta: NULL argument"); return LO_EINVAL; }
    if (!f->cas || f->n_spin != 2) {
        set_error("lo_set_cas_trial_beta: needs an unrestricted factor set and a preceding lo_set_cas_trial with the alpha strings");
        return LO_EINVAL;
    }
    CasPlan* c = f->cas;
    const int n_orb_b = f->n_occ[1];
    if (n_ref_b <= 0 || n_ref_b > n_orb_b) { set_error("lo_set_cas_trial_beta: n_ref_b out of range"); return LO_EINVAL; }
    lo_status st = check_strings(c->n_det, c->max_exc, n_ref_b, n_orb_b, holes_b, parts_b);
    if (st != LO_OK) return st;
    CK(cudaSetDevice(f->device));
    std::vector<int> act;
    for (size_t k = 0; k < (size_t)c->n_det * c->max_exc; ++k)
        if (holes_b[k] >= 0 && std::find(act.begin(), act.end(), holes_b[k]) == act.end()) act.push_back(holes_b[k]);
    std::sort(act.begin(), act.end());
    if (c->mode == LO_CAS_SMW_ENERGY && act.size() > 6) {
        set_error("lo_set_cas_trial_beta: LO_CAS_SMW_ENERGY supports at most 6 distinct hole columns per spin; use LO_CAS_DIRECT");
        return LO_EINVAL;
    }
    void* old[] = {c->dHolesB, c->dPartsB, c->dTh0B, c->dA0B, c->dTB, c->dGB, c->dWdB, c->dSt0B, c->dHoleIdxB, c->dKindB, c->dSB, c->dHB, c->dPartB,
                   c->dStVB, c->dThAct[1], c->dZ[1], c->dPairs[1], c->dPassAct[1]};
    for (void* q : old)
        if (q) cudaFree(q);
    c->dHolesB = c->dPartsB = nullptr; c->dTh0B = c->dA0B = c->dTB = c->dGB = c->dWdB = nullptr; c->dSt0B = nullptr;
    c->dHoleIdxB = nullptr; c->dKindB = nullptr; c->dSB = c->dHB = c->dPartB = nullptr; c->dStVB = nullptr; c->dThAct[1] = c->dZ[1] = nullptr; c->dPairs[1] = nullptr; c->dPassAct[1] = nullptr;
    c->has_beta = false;
    c->n_ref_b = n_ref_b; c->n_virt_b = n_orb_b - n_ref_b;
    const size_t nv = (size_t)c->max_real * c->n_det, ne = (size_t)c->n_det * c->max_exc;
    auto al = [&](void** p, size_t bytes) -> cudaError_t {
        cudaError_t e = cudaMalloc(p, std::max<size_t>(bytes, 16));
        if (e == cudaSuccess) e = cudaMemset(*p, 0, std::max<size_t>(bytes, 16));
        return e;
    };
    CK(al((void**)&c->dHolesB, ne * 4));
    CK(al((void**)&c->dPartsB, ne * 4));
    CK(al((void**)&c->dTh0B, (size_t)n_orb_b * 2 * c->W0cap * f->N_pad * 8));
    CK(al((void**)&c->dA0B, (size_t)c->W0cap * n_ref_b * n_ref_b * 16));
    CK(al((void**)&c->dTB, (size_t)c->W0cap * std::max(c->n_virt_b, 1) * n_ref_b * 16));
    CK(al((void**)&c->dGB, nv * c->max_exc * n_orb_b * 16));
    CK(al((void**)&c->dWdB, nv * 16));
    CK(al((void**)&c->dSt0B, (size_t)c->W0cap * 4));
    CK(cudaMemcpy(c->dHolesB, holes_b, ne * 4, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(c->dPartsB, parts_b, ne * 4, cudaMemcpyHostToDevice));
    if (c->mode == LO_CAS_SMW_ENERGY) {
        st = alloc_smw_spin(f, c, 1, holes_b, parts_b, act);
        if (st != LO_OK) return st;      // has_beta stays false: lo_local_energy_cas refuses to run
    }
    c->has_beta = true;
    return LO_OK;
}

lo_status lo_local_energy_cas(const lo_factors* fc, int n_w, const void* phi, const void* phi_b, void* E_L, void* E1, void* E_J, void* E_K,
                              void* ovlp, int* walker_status, void* stream) {
    if (!fc || !phi || !E_L) { set_error("lo_local_energy_cas: NULL argument"); return LO_EINVAL; }
    if (fc->cas && fc->n_spin == 2 && (!fc->cas->has_beta || !phi_b || ((uintptr_t)phi_b & 15))) {
        set_error("lo_local_energy_cas: an unrestricted trial needs lo_set_cas_trial_beta and a 16-byte aligned phi_b");
        return LO_EINVAL;
    }
    if (fc->device < 0) { set_error("lo_local_energy_cas: no device; there is no CPU path"); return LO_ECUDA; }
    if (!fc->cas) { set_error("lo_local_energy_cas: call lo_set_cas_trial first"); return LO_EINVAL; }
    if (n_w <= 0 || n_w > fc->cas->max_real || n_w > 65535) { set_error("lo_local_energy_cas: n_w out of range (1..min(max_real_walkers, 65535))"); return LO_EINVAL; }
    if (((uintptr_t)phi & 15) || ((uintptr_t)E_L & 15) || ((uintptr_t)E1 & 15) || ((uintptr_t)E_J & 15) || ((uintptr_t)E_K & 15) || ((uintptr_t)ovlp & 15)) {
        set_error("lo_local_energy_cas: pointers must be 16-byte aligned");
        return LO_EINVAL;
    }
    lo_factors* f = const_cast<lo_factors*>(fc);
    CK(cudaSetDevice(f->device));
    const int ex_mode = f->ex_mode;      // the multi-determinant path keeps its DMMA kernels (lo_set_exchange_mode)
    f->ex_mode = LO_EXCHANGE_DMMA;
    const lo_status st = launch_local_energy_cas(f, n_w, phi, f->n_spin == 2 ? phi_b : nullptr, E_L, E1, E_J, E_K, ovlp, walker_status, (cudaStream_t)stream);
    f->ex_mode = ex_mode;
    return st;
}

lo_status lo_propagator(const lo_factors* fc, int n_w, const void* x_dev, void* stream) {
    if (!fc || !x_dev) { set_error("lo_propagator: NULL argument"); return LO_EINVAL; }
    if (fc->device < 0) { set_error("lo_propagator: no device"); return LO_ECUDA; }
    if (!fc->ops->dLt || !fc->dB) { set_error("lo_propagator: the factor set was built without LO_SETUP_PROPAGATOR"); return LO_EINVAL; }
    if (n_w <= 0 || n_w > fc->max_walkers || n_w > 65535) { set_error("lo_propagator: n_w out of range (1..min(max_walkers, 65535): grid dimension of the field-packing kernel)"); return LO_EINVAL; }
    if ((uintptr_t)x_dev & 15) { set_error("lo_propagator: x must be 16-byte aligned"); return LO_EINVAL; }
    lo_factors* f = const_cast<lo_factors*>(fc);
    CK(cudaSetDevice(f->device));
    return launch_propagator(f, n_w, x_dev, (cudaStream_t)stream);
}

lo_status lo_propagator_buffer(const lo_factors* f, const void** B_dev, int* ld, long long* n_rows) {
    if (!f || !B_dev || !ld || !n_rows) { set_error("lo_propagator_buffer: NULL argument"); return LO_EINVAL; }
    if (f->device < 0 || !f->dB) { set_error("lo_propagator_buffer: the factor set was built without LO_SETUP_PROPAGATOR"); return LO_EINVAL; }
    *B_dev = f->dB;
    *ld = f->Wcap;
    *n_rows = f->ops->tri;
    return LO_OK;
}

lo_status lo_propagator_host(const lo_factors* f, int w, void* B_host) {
    if (!f || !B_host || w < 0 || w >= f->max_walkers) { set_error("lo_propagator_host: invalid argument"); return LO_EINVAL; }
    if (f->device < 0 || !f->dB) { set_error("lo_propagator_host: the factor set was built without LO_SETUP_PROPAGATOR"); return LO_EINVAL; }
    CK(cudaSetDevice(f->device));
    CK(cudaDeviceSynchronize());
    const long long tri = f->ops->tri;
    std::vector<double> col((size_t)tri * 2);
    // column w of complex [tri][Wcap]: 16 bytes per row, pitch ldw*8
    CK(cudaMemcpy2D(col.data(), 16, f->dB + (size_t)2 * w, (size_t)f->ldw * 8, 16, (size_t)tri, cudaMemcpyDeviceToHost));
    double* out = static_cast<double*>(B_host);
    const int N = f->N;
    long long r = 0;
    for (int p = 0; p < N; ++p)
        for (int q = p; q < N; ++q, ++r) {
            out[((size_t)p * N + q) * 2] = out[((size_t)q * N + p) * 2] = col[2 * r];
            out[((size_t)p * N + q) * 2 + 1] = out[((size_t)q * N + p) * 2 + 1] = col[2 * r + 1];
        }
    return LO_OK;
}

lo_status lo_theta_host(const lo_factors* f, int spin, int n_w, void* theta_host) {
    if (!f || !theta_host || spin < 0 || spin >= f->n_spin || n_w <= 0 || n_w > f->max_walkers) { set_error("lo_theta_host: invalid argument"); return LO_EINVAL; }
    if (f->device < 0) { set_error("lo_theta_host: no device"); return LO_ECUDA; }
    CK(cudaSetDevice(f->device));
    CK(cudaDeviceSynchronize());
    const int O = f->n_occ[spin], N = f->N, N_pad = f->N_pad;
    std::vector<double> panel((size_t)2 * n_w * N_pad);
    double* out = static_cast<double*>(theta_host);
    for (int i = 0; i < O; ++i) {
        CK(cudaMemcpy(panel.data(), f->dThT + (size_t)(f->o_base[spin] + i) * f->ldw * N_pad, panel.size() * 8, cudaMemcpyDeviceToHost));
        for (int w = 0; w < n_w; ++w)
            for (int p = 0; p < N; ++p) {
                out[(((size_t)w * N + p) * O + i) * 2] = panel[(size_t)(2 * w) * N_pad + p];
                out[(((size_t)w * N + p) * O + i) * 2 + 1] = panel[(size_t)(2 * w + 1) * N_pad + p];
            }
    }
    return LO_OK;
}

lo_status lo_timing_enable(lo_factors* f, int enable) {
    if (!f) { set_error("lo_timing_enable: NULL"); return LO_EINVAL; }
    f->timing = enable != 0;
    return LO_OK;
}

lo_status lo_timing_get(lo_factors* f, double ms[LO_K_COUNT], long long launches[LO_K_COUNT]) {
    if (!f || !ms || !launches) { set_error("lo_timing_get: NULL"); return LO_EINVAL; }
    if (f->device >= 0) {
        CK(cudaSetDevice(f->device));
        for (auto& ev : f->events) {
            CK(cudaEventSynchronize(ev.e1));
            float t = 0;
            CK(cudaEventElapsedTime(&t, ev.e0, ev.e1));
            f->t_ms[ev.kind] += t;
            f->t_n[ev.kind] += 1;
            f->pool.push_back(ev);
        }
        f->events.clear();
    }
    for (int k = 0; k < LO_K_COUNT; ++k) { ms[k] = f->t_ms[k]; launches[k] = f->t_n[k]; f->t_ms[k] = 0; f->t_n[k] = 0; }
    return LO_OK;
}

lo_status lo_flops_per_walker(const lo_factors* f, double fl[LO_K_COUNT]) {
    if (!f || !fl) { set_error("lo_flops_per_walker: NULL"); return LO_EINVAL; }
    for (int k = 0; k < LO_K_COUNT; ++k) fl[k] = 0;
    const double N = f->N;
    double R = 0;
    for (int s = 0; s < f->n_spin; ++s) {
        const double O = f->n_occ[s];
        fl[LO_K_OVERLAP] += 4.0 * N * O * O;            // real x complex
        fl[LO_K_INVERSE] += 8.0 * O * O * O;            // Gauss-Jordan, complex
        fl[LO_K_THETA] += 8.0 * N * O * O;              // complex x complex
        for (int r : f->rank[s]) R += r;
    }
    fl[LO_K_COULOMB] = 4.0 * (f->n_chol + 1.0) * N * f->O_tot;   // real x complex, incl. the hbar row (S2)
    fl[LO_K_EXCHANGE] = (f->coulomb_lo ? 2.0 : 1.0) * (8.0 * N * R + 8.0 * R);   // two (compressed-Coulomb mode: four) real x complex GEMMs + weighted complex dots
    fl[LO_K_PROPAGATOR] = 4.0 * f->n_chol * (N * (N + 1.0) / 2.0);  // lo_propagator (not part of lo_local_energy): real x complex
    return LO_OK;
}

lo_status lo_measure_peak(int device, int kind, double* value) {
    if (!value) { set_error("lo_measure_peak: NULL"); return LO_EINVAL; }
    return measure_peak(device, kind, value);
}

void lo_free(lo_factors* f) { free_all(f); }

}  // extern "C"
