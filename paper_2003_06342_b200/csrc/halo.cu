// Ghost-layer exchange of slab contexts (include/lbm.h "slab decomposition"; the paper's MPI decomposition, PAPER.md:324,
// 559): pack the boundary layer of one side into a contiguous device buffer / unpack a neighbour's buffer into the ghost
// layer.  One launch each; the transport between the two is the caller's (NCCL send/recv, peer copy, same buffer).
#include "ctx.h"
#include "lattices.cuh"

namespace lbm {

constexpr int HALO_MAX_REGIONS = 12;   // 3 + 3 + 3 of (D2Q9, D2Q9, D2Q9) is the largest set

struct HaloPlan {
    int count;                       // contiguous regions of `elems` elements each
    unsigned long long elems;
    char *ptr[HALO_MAX_REGIONS];     // device address of each region in the workspace
};

// buffer layout: region r occupies [r * elems, (r + 1) * elems)
template <class T>
__global__ void __launch_bounds__(256) k_halo_copy(const HaloPlan plan, T *__restrict__ buf, const int pack) {
    const int r = blockIdx.y;
    T *reg = reinterpret_cast<T *>(plan.ptr[r]);
    T *b = buf + (unsigned long long)r * plan.elems;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < plan.elems;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        if (pack) b[i] = reg[i];
        else reg[i] = b[i];
    }
}

// region r of `src` into region r of `dst` (same number and size of regions): a boundary layer straight into a ghost layer
template <class T>
__global__ void __launch_bounds__(256) k_halo_push(const HaloPlan src, const HaloPlan dst) {
    const int r = blockIdx.y;
    const T *a = reinterpret_cast<const T *>(src.ptr[r]);
    T *b = reinterpret_cast<T *>(dst.ptr[r]);
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < src.elems;
         i += (unsigned long long)gridDim.x * blockDim.x)
        b[i] = a[i];
}

namespace {

template <class L> void add_pops(HaloPlan &pl, const lbm_ctx *c, size_t off, int axis, int dir, long long layer, size_t es) {
    const long long layer_elems = (long long)pl.elems;
    for (int i = 0; i < L::Q; ++i) {
        const int e = axis == 2 ? L::ez(i) : L::ey(i);
        if (e != dir) continue;
        pl.ptr[pl.count++] = c->ws + off + ((size_t)i * (size_t)c->L.N + (size_t)layer * (size_t)layer_elems) * es;
    }
}

// what: LBM_HALO_PHI / LBM_HALO_POPS; side: 0 low, 1 high; ghost: the ghost layer of that side (unpack) or the owned
// boundary layer next to it (pack)
bool make_plan(const lbm_ctx *c, int what, int side, bool ghost, HaloPlan &pl) {
    const lbm_params &P = c->P;
    const bool three_d = P.nz > 1;
    const int axis = three_d ? 2 : 1;
    const int len = three_d ? P.nz : P.ny;
    const size_t es = (size_t)c->L.es, esp = (size_t)c->L.es_phi;
    long long layer = side == 0 ? 0 : len - 1;
    if (!ghost) layer += side == 0 ? 1 : -1;
    pl.count = 0;
    if (what == LBM_HALO_PHI) {
        // padded array: layer l of the domain is padded layer l + 1 along the slab axis; whole padded layer with its images
        const size_t layer_elems = three_d ? (size_t)c->L.ppx * c->L.ppy : (size_t)c->L.ppx;
        pl.elems = layer_elems;
        // between the phases -- and while parts of phase 0 are running (lbm_step_layers) -- phi^{n+1} is the other buffer
        const int pnew = (c->phase == 1 || c->partial) ? 1 - c->curphi : c->curphi;
        pl.ptr[pl.count++] = c->ws + c->L.off_phi[pnew] + (size_t)(layer + 1) * layer_elems * esp;
        return true;
    }
    // populations that stream across the cut towards `side`: e_axis = +1 for the high side, -1 for the low side.
    // A ghost layer of side s RECEIVES what the neighbour sent towards its 1 - s side, i.e. e_axis pointing inwards.
    const int dir = ghost ? (side == 0 ? +1 : -1) : (side == 0 ? -1 : +1);
    pl.elems = three_d ? (unsigned long long)P.nx * P.ny : (unsigned long long)P.nx;
    // the populations of the level just collided: the current buffers, or -- while parts of phase 1 are running and the
    // buffers have not flipped yet (lbm_step_layers) -- the other ones
    const int cur = (c->phase == 1 && c->partial) ? 1 - c->cur : c->cur;
    switch (c->set) {
    case SET_2D_995:
        add_pops<D2Q9>(pl, c, c->L.off_f[cur], axis, dir, layer, es);
        add_pops<D2Q9>(pl, c, c->L.off_g[cur], axis, dir, layer, es);
        add_pops<D2Q5>(pl, c, c->L.off_s[cur], axis, dir, layer, es);
        break;
    case SET_2D_999:
        add_pops<D2Q9>(pl, c, c->L.off_f[cur], axis, dir, layer, es);
        add_pops<D2Q9>(pl, c, c->L.off_g[cur], axis, dir, layer, es);
        add_pops<D2Q9>(pl, c, c->L.off_s[cur], axis, dir, layer, es);
        break;
    case SET_3D_1977:
        add_pops<D3Q19>(pl, c, c->L.off_f[cur], axis, dir, layer, es);
        add_pops<D3Q7>(pl, c, c->L.off_g[cur], axis, dir, layer, es);
        add_pops<D3Q7>(pl, c, c->L.off_s[cur], axis, dir, layer, es);
        break;
    case SET_3D_1577:
        add_pops<D3Q15>(pl, c, c->L.off_f[cur], axis, dir, layer, es);
        add_pops<D3Q7>(pl, c, c->L.off_g[cur], axis, dir, layer, es);
        add_pops<D3Q7>(pl, c, c->L.off_s[cur], axis, dir, layer, es);
        break;
    default: return false;
    }
    return pl.count > 0 && pl.count <= HALO_MAX_REGIONS;
}

int halo_copy(lbm_ctx *c, int what, int side, void *d_buf, bool pack) {
    if (!c || !d_buf || (what != LBM_HALO_PHI && what != LBM_HALO_POPS) || (side != 0 && side != 1)) return LBM_E_INVALID;
    if (!c->P.halo[side]) return LBM_E_INVALID;
    if (!c->inited) return LBM_E_STATE;
    // phi travels between the phases or while parts of phase 0 are running; the populations after phase 1 (or after lbm_init)
    // or while parts of phase 1 are running (lbm_step_layers: boundary layers first)
    const bool phi_time = (c->phase == 1 && !c->partial) || (c->phase == 0 && c->partial);
    if ((what == LBM_HALO_PHI) != phi_time) return LBM_E_STATE;
    HaloPlan pl;
    if (!make_plan(c, what, side, /*ghost=*/!pack, pl)) return LBM_E_INVALID;
    const unsigned gx = (unsigned)((pl.elems + 1023) / 1024 > 0 ? (pl.elems + 1023) / 1024 : 1);
    const dim3 grid(gx > 1184u ? 1184u : gx, (unsigned)pl.count);
    if ((what == LBM_HALO_PHI ? c->L.es_phi : c->L.es) == 8) k_halo_copy<double><<<grid, 256, 0, c->stream>>>(pl, static_cast<double *>(d_buf), pack ? 1 : 0);
    else k_halo_copy<float><<<grid, 256, 0, c->stream>>>(pl, static_cast<float *>(d_buf), pack ? 1 : 0);
    c->launches++;
    CK(cudaGetLastError());
    return LBM_OK;
}

}  // namespace
}  // namespace lbm

extern "C" {

int lbm_halo_bytes(const lbm_ctx *c, int what, size_t *bytes) {
    if (!c || !bytes || (what != LBM_HALO_PHI && what != LBM_HALO_POPS)) return LBM_E_INVALID;
    if (!(c->P.halo[0] | c->P.halo[1])) return LBM_E_INVALID;
    lbm::HaloPlan pl;
    const int side = c->P.halo[0] ? 0 : 1;   // the size depends neither on the side nor on the phase
    if (!lbm::make_plan(c, what, side, false, pl)) return LBM_E_INVALID;
    *bytes = (size_t)pl.count * (size_t)pl.elems * (size_t)(what == LBM_HALO_PHI ? c->L.es_phi : c->L.es);
    return LBM_OK;
}

namespace lbm {
namespace {
// boundary layer of `side` of c -> ghost layer of the opposite side of `peer` (a context, or a description of a mapped workspace)
int halo_push(lbm_ctx *c, int what, int side, const lbm_ctx *peer);
}  // namespace
}  // namespace lbm

int lbm_halo_push(lbm_ctx *c, int what, int side, lbm_ctx *peer) {
    if (!c || !peer) return LBM_E_INVALID;
    if (!peer->inited) return LBM_E_STATE;
    // both contexts at the same point of the same step (see halo_copy for when phi and when the populations travel)
    if (c->phase != peer->phase || c->partial != peer->partial || c->cur != peer->cur || c->curphi != peer->curphi) return LBM_E_STATE;
    return lbm::halo_push(c, what, side, peer);
}

int lbm_halo_push_mapped(lbm_ctx *c, int what, int side, const lbm_params *peer_params, void *d_peer_workspace) {
    using namespace lbm;
    if (!c || !peer_params || !d_peer_workspace) return LBM_E_INVALID;
    // a description of the neighbour's context, standing where this one stands: the two step in lockstep
    lbm_ctx peer{};
    const int rc = describe_params(peer_params, &peer.set, &peer.L);
    if (rc) return rc;
    peer.P = *peer_params;
    peer.ws = static_cast<char *>(d_peer_workspace);
    peer.inited = true; peer.phase = c->phase; peer.partial = c->partial; peer.cur = c->cur; peer.curphi = c->curphi;
    return halo_push(c, what, side, &peer);
}

namespace lbm {
namespace {
int halo_push(lbm_ctx *c, int what, int side, const lbm_ctx *peer) {
    if ((what != LBM_HALO_PHI && what != LBM_HALO_POPS) || (side != 0 && side != 1)) return LBM_E_INVALID;
    if (!c->P.halo[side] || !peer->P.halo[1 - side]) return LBM_E_INVALID;
    if (!c->inited) return LBM_E_STATE;
    const bool phi_time = (c->phase == 1 && !c->partial) || (c->phase == 0 && c->partial);
    if ((what == LBM_HALO_PHI) != phi_time) return LBM_E_STATE;
    if (c->set != peer->set || c->L.es != peer->L.es || c->P.nx != peer->P.nx || (c->P.nz > 1 && c->P.ny != peer->P.ny)) return LBM_E_INVALID;
    HaloPlan src, dst;
    if (!make_plan(c, what, side, /*ghost=*/false, src) || !make_plan(peer, what, 1 - side, /*ghost=*/true, dst)) return LBM_E_INVALID;
    if (src.count != dst.count || src.elems != dst.elems) return LBM_E_INVALID;   // the two slabs differ in the slab axis only
    const unsigned gx = (unsigned)((src.elems + 1023) / 1024 > 0 ? (src.elems + 1023) / 1024 : 1);
    const dim3 grid(gx > 1184u ? 1184u : gx, (unsigned)src.count);
    if ((what == LBM_HALO_PHI ? c->L.es_phi : c->L.es) == 8) k_halo_push<double><<<grid, 256, 0, c->stream>>>(src, dst);
    else k_halo_push<float><<<grid, 256, 0, c->stream>>>(src, dst);
    c->launches++;
    CK(cudaGetLastError());
    return LBM_OK;
}
}  // namespace
}  // namespace lbm

int lbm_halo_pack(lbm_ctx *c, int what, int side, void *d_buf) { return lbm::halo_copy(c, what, side, d_buf, true); }

int lbm_halo_unpack(lbm_ctx *c, int what, int side, const void *d_buf) {
    return lbm::halo_copy(c, what, side, const_cast<void *>(d_buf), false);
}

}  // extern "C"

// ---- stream-ordered flags for the peer transport (include/lbm.h): cuStreamWriteValue32 / cuStreamWaitValue32 are executed by the
// GPU's front end in stream order -- no kernel spins, no host call waits -- and the write is a memory barrier for everything the
// stream did before it, so a counter written into the neighbour's (peer-mapped) memory after a push says "the ghost layer is there".
#include <cudaTypedefs.h>

namespace {
typedef CUresult(CUDAAPI *stream_value_fn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
stream_value_fn stream_value_entry(const char *name) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) return nullptr;
    return reinterpret_cast<stream_value_fn>(p);
}
}  // namespace

extern "C" int lbm_stream_signal(lbm_ctx *c, void *d_flag, unsigned value) {
    if (!c || !d_flag) return LBM_E_INVALID;
    static stream_value_fn fn = stream_value_entry("cuStreamWriteValue32");
    if (!fn) return LBM_E_UNSUPPORTED;
    if (fn(c->stream, reinterpret_cast<CUdeviceptr>(d_flag), value, CU_STREAM_WRITE_VALUE_DEFAULT) != CUDA_SUCCESS) return LBM_E_CUDA;
    return LBM_OK;
}

extern "C" int lbm_stream_wait(lbm_ctx *c, void *d_flag, unsigned value) {
    if (!c || !d_flag) return LBM_E_INVALID;
    static stream_value_fn fn = stream_value_entry("cuStreamWaitValue32");
    if (!fn) return LBM_E_UNSUPPORTED;
    if (fn(c->stream, reinterpret_cast<CUdeviceptr>(d_flag), value, CU_STREAM_WAIT_VALUE_GEQ) != CUDA_SUCCESS) return LBM_E_CUDA;
    return LBM_OK;
}
