// Checkpoint / resume (include/lbm.h): the whole state of a context -- its workspace and the few host-side counters that say which
// of the double buffers hold the current level -- to and from one HOST buffer.  A restored context continues bit for bit.
#include "ctx.h"

#include <cstring>

namespace {
struct StateHeader {           // 64 bytes in front of the workspace image
    unsigned long long magic;  // "LBMSTATE"
    unsigned long long workspace_bytes;
    long long nsteps;
    int cur, curphi, phase, precision;
    int nx, ny, nz, lattice_set;
    unsigned long long pad;
};
static_assert(sizeof(StateHeader) == 64, "header layout");
constexpr unsigned long long MAGIC = 0x45544154534d424cULL;   // 'LBMSTATE', little endian
}  // namespace

extern "C" size_t lbm_state_bytes(const lbm_ctx *c) { return c ? sizeof(StateHeader) + c->L.total : 0; }

extern "C" int lbm_save_state(lbm_ctx *c, void *h_state) {
    using namespace lbm;
    if (!c || !h_state) return LBM_E_INVALID;
    if (!c->inited || c->phase != 0 || c->partial) return LBM_E_STATE;   // between steps only
    StateHeader h{};
    h.magic = MAGIC; h.workspace_bytes = c->L.total; h.nsteps = c->nsteps;
    h.cur = c->cur; h.curphi = c->curphi; h.phase = c->phase; h.precision = c->P.precision;
    h.nx = c->P.nx; h.ny = c->P.ny; h.nz = c->P.nz; h.lattice_set = (int)c->set;
    std::memcpy(h_state, &h, sizeof(h));
    CK(cudaMemcpyAsync(static_cast<char *>(h_state) + sizeof(h), c->ws, c->L.total, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return LBM_OK;
}

extern "C" int lbm_load_state(lbm_ctx *c, const void *h_state) {
    using namespace lbm;
    if (!c || !h_state) return LBM_E_INVALID;
    StateHeader h;
    std::memcpy(&h, h_state, sizeof(h));
    // the image must come from a context of the same grid, lattice set and precision (the physical parameters are the caller's)
    if (h.magic != MAGIC || h.workspace_bytes != c->L.total || h.precision != c->P.precision || h.nx != c->P.nx || h.ny != c->P.ny ||
        h.nz != c->P.nz || h.lattice_set != (int)c->set || (h.cur | 1) != 1 || (h.curphi | 1) != 1 || h.phase != 0)
        return LBM_E_INVALID;
    CK(cudaMemcpyAsync(c->ws, static_cast<const char *>(h_state) + sizeof(h), c->L.total, cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    c->cur = h.cur; c->curphi = h.curphi; c->phase = 0; c->partial = false; c->nsteps = h.nsteps; c->inited = true;
    return LBM_OK;
}
