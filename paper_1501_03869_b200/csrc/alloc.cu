// alloc.cu -- the ONLY place where the library obtains or returns device memory on its own.
//
// device memory belongs to the caller.  The big, size-predictable part is the workspace handed to
// pat_plan_create.  Everything whose size depends on the data -- work lists, the optional weight table, geometry
// for the conventional BP, the ROI-masked permutation, scratch of the set-up kernels and of the eikonal solver --
// is requested through a provider the caller installs with pat_set_device_allocator (the Python binding installs
// one that hands out torch tensors).  Without a provider the shim below falls back to cudaMalloc / cudaFree.
#include "pat_internal.h"

#include <cuda_runtime.h>

#include <mutex>

namespace {
std::mutex g_alloc_mu;
PatAllocator g_alloc;                      // process-wide provider (all NULL = built-in cudaMalloc shim)
}  // namespace

extern "C" pat_status pat_set_device_allocator(pat_alloc_fn alloc, pat_free_fn release, void *user) {
    if ((alloc == nullptr) != (release == nullptr)) return PAT_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lk(g_alloc_mu);
    g_alloc.alloc = alloc;
    g_alloc.release = release;
    g_alloc.user = user;
    return PAT_OK;
}

PatAllocator pat_current_allocator() {
    std::lock_guard<std::mutex> lk(g_alloc_mu);
    return g_alloc;
}

bool pat_dev_alloc(const PatAllocator &a, size_t bytes, PatDevBuf *out, int64_t *held, int64_t *peak) {
    out->p = nullptr;
    out->bytes = 0;
    if (bytes == 0) bytes = 256;
    void *ptr = nullptr;
    if (a.alloc) {
        ptr = a.alloc(bytes, a.user);
        if (ptr && (((uintptr_t)ptr) & 255u)) {        // a provider must return 256-byte aligned device memory
            a.release(ptr, bytes, a.user);
            ptr = nullptr;
        }
    } else {
        if (cudaMalloc(&ptr, bytes) != cudaSuccess) { cudaGetLastError(); ptr = nullptr; }
    }
    if (!ptr) return false;
    out->p = ptr;
    out->bytes = bytes;
    if (held) {
        *held += (int64_t)bytes;
        if (peak && *held > *peak) *peak = *held;
    }
    return true;
}

void pat_dev_free(const PatAllocator &a, PatDevBuf *buf, int64_t *held) {
    if (!buf->p) return;
    if (a.release) a.release(buf->p, buf->bytes, a.user);
    else cudaFree(buf->p);
    if (held) *held -= (int64_t)buf->bytes;
    buf->p = nullptr;
    buf->bytes = 0;
}
