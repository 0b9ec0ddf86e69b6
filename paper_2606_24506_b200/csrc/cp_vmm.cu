// cp_vmm.cu -- CUDA virtual memory management behind the arena.
//
// One virtual range is reserved for the whole pool and cut into one slot per request id; a slot is
// a request's contiguous virtual KV space.  Physical memory comes in chunks of the device's
// allocation granularity; a chunk is created the first time it is needed, mapped where a request
// grows into it, and parked (still allocated, mapped nowhere) when the request finishes, so that a
// later mapping costs cuMemMap + cuMemSetAccess only.  The number of chunks that exist never
// exceeds the budget: that is the pool page budget of the paper, in physical terms.
#include "cp_vmm.h"

#include <cuda.h>
#include <cuda_runtime.h>
#include <new>

namespace cp {

namespace {

struct DriverApi {
    CUresult (*AddressReserve)(CUdeviceptr *, size_t, size_t, CUdeviceptr, unsigned long long) = nullptr;
    CUresult (*AddressFree)(CUdeviceptr, size_t) = nullptr;
    CUresult (*Create)(CUmemGenericAllocationHandle *, size_t, const CUmemAllocationProp *, unsigned long long) = nullptr;
    CUresult (*Release)(CUmemGenericAllocationHandle) = nullptr;
    CUresult (*Map)(CUdeviceptr, size_t, size_t, CUmemGenericAllocationHandle, unsigned long long) = nullptr;
    CUresult (*Unmap)(CUdeviceptr, size_t) = nullptr;
    CUresult (*SetAccess)(CUdeviceptr, size_t, const CUmemAccessDesc *, size_t) = nullptr;
    CUresult (*GetGranularity)(size_t *, const CUmemAllocationProp *, CUmemAllocationGranularity_flags) = nullptr;
    bool ok = false;
};

template <typename F>
bool fetch(const char *name, F *fn)
{
    void *ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint(name, &ptr, cudaEnableDefault, &q) != cudaSuccess || !ptr ||
        q != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    *fn = reinterpret_cast<F>(ptr);
    return true;
}

const DriverApi &driver()
{
    static DriverApi api = [] {
        DriverApi a;
        a.ok = fetch("cuMemAddressReserve", &a.AddressReserve) && fetch("cuMemAddressFree", &a.AddressFree) &&
               fetch("cuMemCreate", &a.Create) && fetch("cuMemRelease", &a.Release) && fetch("cuMemMap", &a.Map) &&
               fetch("cuMemUnmap", &a.Unmap) && fetch("cuMemSetAccess", &a.SetAccess) &&
               fetch("cuMemGetAllocationGranularity", &a.GetGranularity);
        return a;
    }();
    return api;
}

CUmemAllocationProp device_prop(int device)
{
    CUmemAllocationProp prop = {};
    prop.type = CU_MEM_ALLOCATION_TYPE_PINNED;
    prop.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    prop.location.id = device;
    return prop;
}

uint64_t round_up(uint64_t x, uint64_t m) { return (x + m - 1) / m * m; }

uint64_t gcd_u64(uint64_t a, uint64_t b)
{
    while (b) { const uint64_t t = a % b; a = b; b = t; }
    return a;
}

}  // namespace

int vmm_create(VmmArena **out, uint64_t slot_bytes_min, int n_slots, uint64_t budget_bytes, uint64_t slot_align_bytes)
{
    *out = nullptr;
    int device = 0;
    if (cudaFree(nullptr) != cudaSuccess || cudaGetDevice(&device) != cudaSuccess) {   // also creates the context
        cudaGetLastError();
        return 1;
    }
    const DriverApi &api = driver();
    if (!api.ok) return 1;
    const CUmemAllocationProp prop = device_prop(device);
    size_t gran = 0;
    if (api.GetGranularity(&gran, &prop, CU_MEM_ALLOC_GRANULARITY_MINIMUM) != CUDA_SUCCESS || gran == 0) return 2;
    VmmArena *a = new (std::nothrow) VmmArena();
    if (!a) return 2;
    a->device = device;
    a->chunk_bytes = gran;
    // a slot starts on a chunk boundary AND on a page boundary (page ids are plain arithmetic)
    const uint64_t unit = gran / gcd_u64(gran, slot_align_bytes) * slot_align_bytes;
    a->slot_bytes = round_up(slot_bytes_min, unit);
    a->n_slots = n_slots;
    a->va_bytes = a->slot_bytes * (uint64_t)n_slots;
    a->budget_chunks = (uint32_t)(budget_bytes / gran);
    a->slot_chunks.resize(n_slots);
    CUdeviceptr base = 0;
    // page k sits at base + k * page_bytes: the base itself needs the default (chunk) alignment only
    if (api.AddressReserve(&base, a->va_bytes, 0, 0, 0) != CUDA_SUCCESS) {
        delete a;
        return 2;
    }
    a->base = (uint64_t)base;
    *out = a;
    return 0;
}

void vmm_destroy(VmmArena *a)
{
    if (!a) return;
    const DriverApi &api = driver();
    for (int s = 0; s < a->n_slots; ++s) vmm_release_slot(a, s);
    for (uint64_t h : a->parked) api.Release((CUmemGenericAllocationHandle)h);
    if (a->base) api.AddressFree((CUdeviceptr)a->base, a->va_bytes);
    delete a;
}

uint32_t vmm_chunks_missing(const VmmArena *a, int slot, uint64_t bytes)
{
    const uint64_t want = (bytes + a->chunk_bytes - 1) / a->chunk_bytes;
    const uint64_t have = a->slot_chunks[slot].size();
    return want > have ? (uint32_t)(want - have) : 0;
}

uint32_t vmm_chunks_available(const VmmArena *a)
{
    return (uint32_t)a->parked.size() + (a->budget_chunks - a->created_chunks);
}

uint32_t vmm_chunks_mapped(const VmmArena *a) { return a->created_chunks - (uint32_t)a->parked.size(); }

int vmm_back(VmmArena *a, int slot, uint64_t bytes)
{
    if (bytes > a->slot_bytes) return 3;
    const uint32_t missing = vmm_chunks_missing(a, slot, bytes);
    if (missing == 0) return 0;
    if (missing > vmm_chunks_available(a)) return 3;
    const DriverApi &api = driver();
    const CUmemAllocationProp prop = device_prop(a->device);
    CUmemAccessDesc acc = {};
    acc.location = prop.location;
    acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
    std::vector<uint64_t> &mapped = a->slot_chunks[slot];
    const size_t had = mapped.size();
    const CUdeviceptr va0 = (CUdeviceptr)(a->base + (uint64_t)slot * a->slot_bytes + had * a->chunk_bytes);
    int rc = 0;
    for (uint32_t i = 0; i < missing && rc == 0; ++i) {
        CUmemGenericAllocationHandle h;
        if (!a->parked.empty()) {
            h = (CUmemGenericAllocationHandle)a->parked.back();
            a->parked.pop_back();
        } else {
            if (api.Create(&h, a->chunk_bytes, &prop, 0) != CUDA_SUCCESS) { rc = 2; break; }
            a->created_chunks++;
            a->n_create_calls++;
        }
        if (api.Map(va0 + (uint64_t)i * a->chunk_bytes, a->chunk_bytes, 0, h, 0) != CUDA_SUCCESS) {
            a->parked.push_back((uint64_t)h);
            rc = 2;
            break;
        }
        mapped.push_back((uint64_t)h);
        a->n_map_calls++;
    }
    // one access call for the whole new range
    if (rc == 0 && api.SetAccess(va0, (mapped.size() - had) * a->chunk_bytes, &acc, 1) != CUDA_SUCCESS) rc = 2;
    if (rc != 0) {                                   // undo: the slot keeps the prefix it had
        while (mapped.size() > had) {
            api.Unmap(va0 + (uint64_t)(mapped.size() - 1 - had) * a->chunk_bytes, a->chunk_bytes);
            a->parked.push_back(mapped.back());
            mapped.pop_back();
        }
    }
    return rc;
}

int vmm_release_slot(VmmArena *a, int slot)
{
    std::vector<uint64_t> &mapped = a->slot_chunks[slot];
    if (mapped.empty()) return 0;
    const DriverApi &api = driver();
    const CUdeviceptr va = (CUdeviceptr)(a->base + (uint64_t)slot * a->slot_bytes);
    int rc = 0;
    // one call unmaps the whole backed prefix of the slot (whole mappings only, which these are)
    if (api.Unmap(va, mapped.size() * a->chunk_bytes) != CUDA_SUCCESS) rc = 2;
    for (uint64_t h : mapped) a->parked.push_back(h);
    mapped.clear();
    return rc;
}

}  // namespace cp
