// lbm_read_pops_noalloc (include/lbm.h): lbm_read_pops with its temporary in a file-scope static __device__ array instead of
// cudaMalloc, for callers that must not allocate.  Nothing in this file (or in what it calls) allocates or frees device memory.
#include "ctx.h"

#include <mutex>

namespace {

// One array per GPU that loads the library, held until the process exits.  Shared by every context of the device; keeps the
// last call's contents (the kernel overwrites all it reads back, so nothing has to be cleared).
static __device__ __align__(256) unsigned char g_pops_scratch[LBM_NOALLOC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
void *g_scratch_addr[MAX_DEVICES];   // device address of g_pops_scratch per device, resolved once
std::mutex g_scratch_mutex;

// In host code `g_pops_scratch` is a host-side stand-in, not a device address: the address on the CURRENT device comes from
// cudaGetSymbolAddress, once per device.
int scratch_address(void **out) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return LBM_E_NODEVICE;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        void *p = nullptr;
        CK(cudaGetSymbolAddress(&p, g_pops_scratch));
        if (!p) return LBM_E_CUDA;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return LBM_OK;
}

}  // namespace

extern "C" int lbm_read_pops_noalloc(lbm_ctx *c, int which, int stage, void *h_pops) {
    if (!c || !h_pops || which < 0 || which > 2 || (stage != LBM_STAGE_POSTCOLLISION && stage != LBM_STAGE_STREAMED))
        return LBM_E_INVALID;
    if (!c->inited) return LBM_E_STATE;
    void *d_scratch = nullptr;
    const int rc = scratch_address(&d_scratch);
    if (rc) return rc;
    return c->ops->read_pops_scratch(c, which, stage, h_pops, d_scratch, (size_t)LBM_NOALLOC_SCRATCH_BYTES);
}
