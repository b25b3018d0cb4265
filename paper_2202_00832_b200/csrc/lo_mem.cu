// lo_mem.cu -- growable device arrays with one contiguous virtual address range (CUDA virtual memory management).
//
// lo_setup does not know the size of the packed factor arrays (sum of the truncated ranks, Eq. 18) until the last
// pair block has been decomposed, and at the cage-sized config they reach 2 x 34 GB of the 180 GB of HBM3e: a
// "cudaMalloc the upper bound, then copy to an exact allocation" scheme would double the peak.  GrowBuf reserves the
// upper bound as address space only and maps physical memory chunk by chunk as rows are appended, so the arrays are
// written once, in place, and TMA tensor maps can be encoded over the final contiguous range.
#include <cuda.h>

#include <algorithm>

#include "lo_internal.h"

namespace lo {
namespace {

struct VmmApi {
    CUresult (*AddressReserve)(CUdeviceptr*, size_t, size_t, CUdeviceptr, unsigned long long) = nullptr;
    CUresult (*AddressFree)(CUdeviceptr, size_t) = nullptr;
    CUresult (*Create)(CUmemGenericAllocationHandle*, size_t, const CUmemAllocationProp*, unsigned long long) = nullptr;
    CUresult (*Release)(CUmemGenericAllocationHandle) = nullptr;
    CUresult (*Map)(CUdeviceptr, size_t, size_t, CUmemGenericAllocationHandle, unsigned long long) = nullptr;
    CUresult (*Unmap)(CUdeviceptr, size_t) = nullptr;
    CUresult (*SetAccess)(CUdeviceptr, size_t, const CUmemAccessDesc*, size_t) = nullptr;
    CUresult (*Granularity)(size_t*, const CUmemAllocationProp*, CUmemAllocationGranularity_flags) = nullptr;
    bool ok = false;
};

template <class F>
bool load(const char* name, F& fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !p) return false;
    fn = reinterpret_cast<F>(p);
    return true;
}

VmmApi& api() {
    static VmmApi a;
    static bool tried = false;
    if (!tried) {
        tried = true;
        a.ok = load("cuMemAddressReserve", a.AddressReserve) && load("cuMemAddressFree", a.AddressFree) && load("cuMemCreate", a.Create) &&
               load("cuMemRelease", a.Release) && load("cuMemMap", a.Map) && load("cuMemUnmap", a.Unmap) &&
               load("cuMemSetAccess", a.SetAccess) && load("cuMemGetAllocationGranularity", a.Granularity);
    }
    return a;
}

CUmemAllocationProp prop_for(int device) {
    CUmemAllocationProp p = {};
    p.type = CU_MEM_ALLOCATION_TYPE_PINNED;
    p.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    p.location.id = device;
    return p;
}

}  // namespace

lo_status GrowBuf::reserve(int dev, size_t max_bytes) {
    VmmApi& a = api();
    if (!a.ok) { set_error("CUDA virtual memory management entry points are not available from the driver"); return LO_ECUDA; }
    device = dev;
    CUmemAllocationProp p = prop_for(dev);
    size_t g = 0;
    if (a.Granularity(&g, &p, CU_MEM_ALLOC_GRANULARITY_MINIMUM) != CUDA_SUCCESS || g == 0) { set_error("cuMemGetAllocationGranularity failed"); return LO_ECUDA; }
    chunk = std::max<size_t>(g, (size_t)256 << 20) / g * g;   // 256 MB physical chunks (a multiple of the granularity)
    reserved = (std::max<size_t>(max_bytes, 1) + chunk - 1) / chunk * chunk;
    CUdeviceptr ptr = 0;
    CUresult r = a.AddressReserve(&ptr, reserved, 0, 0, 0);
    if (r != CUDA_SUCCESS) { set_error("cuMemAddressReserve(" + std::to_string(reserved) + " bytes) failed with CUresult " + std::to_string((int)r)); return LO_ENOMEM; }
    base = reinterpret_cast<void*>(ptr);
    mapped = 0;
    return LO_OK;
}

// Make [0, bytes) usable; newly mapped memory is zero-filled (padding rows of the factor arrays rely on it).
lo_status GrowBuf::ensure(size_t bytes) {
    if (bytes <= mapped) return LO_OK;
    if (bytes > reserved) { set_error("GrowBuf: request exceeds the reserved address range"); return LO_EINTERNAL; }
    VmmApi& a = api();
    CUmemAllocationProp p = prop_for(device);
    CUmemAccessDesc acc = {};
    acc.location = p.location;
    acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
    const size_t old = mapped;
    while (mapped < bytes) {
        CUmemGenericAllocationHandle h;
        CUresult r = a.Create(&h, chunk, &p, 0);
        if (r != CUDA_SUCCESS) { set_error("cuMemCreate failed with CUresult " + std::to_string((int)r) + " (out of device memory while growing the factor arrays)"); return LO_ENOMEM; }
        CUdeviceptr at = reinterpret_cast<CUdeviceptr>(base) + mapped;
        r = a.Map(at, chunk, 0, h, 0);
        if (r == CUDA_SUCCESS) r = a.SetAccess(at, chunk, &acc, 1);
        if (r != CUDA_SUCCESS) { a.Release(h); set_error("cuMemMap/cuMemSetAccess failed with CUresult " + std::to_string((int)r)); return LO_ECUDA; }
        handles.push_back((unsigned long long)h);
        mapped += chunk;
    }
    cudaError_t e = cudaMemset(static_cast<char*>(base) + old, 0, mapped - old);
    if (e != cudaSuccess) { set_error(std::string("cudaMemset of newly mapped factor memory: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

void GrowBuf::release() {
    if (!base) return;
    VmmApi& a = api();
    cudaSetDevice(device);
    cudaDeviceSynchronize();
    if (mapped) a.Unmap(reinterpret_cast<CUdeviceptr>(base), mapped);
    for (unsigned long long h : handles) a.Release((CUmemGenericAllocationHandle)h);
    a.AddressFree(reinterpret_cast<CUdeviceptr>(base), reserved);
    handles.clear();
    base = nullptr;
    mapped = reserved = 0;
}

}  // namespace lo
