// cp_vmm.h -- CUDA-VMM-backed arena: one reserved virtual range cut into
// per-request slots, physical chunks mapped on demand ("reserve a virtual KV
// address range ... and map physical KV pages on demand"; mapping is the allocator's slow path).
// Host only.  The driver entry points are fetched at run time (the library does not link libcuda,
// so it still loads on a host without a driver).
#pragma once
#include <cstdint>
#include <vector>

namespace cp {

struct VmmArena {
    uint64_t base = 0;                 // device virtual address of slot 0
    uint64_t va_bytes = 0;             // n_slots * slot_bytes
    uint64_t chunk_bytes = 0;          // allocation granularity (2 MiB on B200)
    uint64_t slot_bytes = 0;           // multiple of chunk_bytes
    int n_slots = 0;
    int device = 0;
    uint32_t budget_chunks = 0;        // physical budget ("pool page budget", in chunks)
    uint32_t created_chunks = 0;       // physical chunks that exist (mapped + parked)
    std::vector<uint64_t> parked;      // handles of physical chunks not mapped anywhere
    std::vector<std::vector<uint64_t>> slot_chunks;   // per slot: handles mapped at chunk 0, 1, ...
    uint64_t n_map_calls = 0, n_create_calls = 0;
};

// 0 = ok, 1 = no usable driver / device, 2 = driver call failed.
int vmm_create(VmmArena **out, uint64_t slot_bytes_min, int n_slots, uint64_t budget_bytes, uint64_t slot_align_bytes);
void vmm_destroy(VmmArena *a);

// Chunks that backing bytes [0, bytes) of `slot` would add.
uint32_t vmm_chunks_missing(const VmmArena *a, int slot, uint64_t bytes);
// Chunks still available (parked + not yet created within the budget).
uint32_t vmm_chunks_available(const VmmArena *a);
uint32_t vmm_chunks_mapped(const VmmArena *a);
// Back bytes [0, bytes) of `slot` (no-op where already backed).  0 = ok, 2 = driver call failed,
// 3 = budget exhausted (nothing changed).
int vmm_back(VmmArena *a, int slot, uint64_t bytes);
// Unmap every chunk of `slot` and park the physical memory for reuse.
int vmm_release_slot(VmmArena *a, int slot);

}  // namespace cp
