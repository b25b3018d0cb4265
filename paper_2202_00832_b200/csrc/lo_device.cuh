// lo_device.cuh -- device helpers shared by the kernel files of liblo_afqmc.so: the DMMA.8x8x4 wrapper, TMA / mbarrier /
// cp.async plumbing, the swizzled fragment addressing, complex helpers and the per-kernel event timer.  Everything sits in an
// anonymous namespace (one copy per translation unit).
#pragma once
#include <cuda.h>

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


constexpr int EX_RING = 8;      // tile-descriptor ring (producer -> consumers), more items than stages can never be in flight

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

}  // namespace
}  // namespace lo
