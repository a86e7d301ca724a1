// lbm_check_finite (include/lbm.h): how many values of the current state are not finite.  Off the hot path: an explicit time
// iteration can leave the stable range (the paper warns of it at low mobility; config 3 of BASELINE.json does
// so after about 10^4 steps), and lbm_step itself never looks.  One counting kernel per array, no allocation: the counter is
// the first 8 bytes of the context's scratch field.
#include "ctx.h"

namespace lbm {

template <class T>
__global__ void __launch_bounds__(256) k_count_nonfinite(const T *__restrict__ a, unsigned long long n, unsigned long long *counter) {
    unsigned long long bad = 0;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (unsigned long long)gridDim.x * blockDim.x)
        bad += isfinite(a[i]) ? 0u : 1u;
    for (int o = 16; o > 0; o >>= 1) bad += __shfl_down_sync(0xffffffffu, bad, o);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(counter, bad);
}

namespace {
template <class T> int count_array(lbm_ctx *c, size_t off, size_t n, unsigned long long *counter) {
    if (!n) return LBM_OK;
    const unsigned blocks = (unsigned)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
    k_count_nonfinite<T><<<blocks, 256, 0, c->stream>>>(reinterpret_cast<const T *>(c->ws + off), (unsigned long long)n, counter);
    c->launches++;
    CK(cudaGetLastError());
    return LBM_OK;
}
}  // namespace

}  // namespace lbm

extern "C" int lbm_check_finite(lbm_ctx *c, long long *n_bad) {
    using namespace lbm;
    if (!c || !n_bad) return LBM_E_INVALID;
    if (!c->inited) return LBM_E_STATE;
    if ((size_t)c->L.N * (size_t)c->L.es < sizeof(unsigned long long)) return LBM_E_UNSUPPORTED;
    auto *counter = reinterpret_cast<unsigned long long *>(c->ws + c->L.off_scratch);
    CK(cudaMemsetAsync(counter, 0, sizeof(unsigned long long), c->stream));
    const size_t N = (size_t)c->L.N;
    const int qf = c->P.lat_f == LBM_D3Q19 ? 19 : (c->P.lat_f == LBM_D3Q15 ? 15 : 9);
    const int qg = c->P.lat_g == LBM_D3Q7 ? 7 : 9;
    const int qs = c->P.lat_s == LBM_D3Q7 ? 7 : (c->P.lat_s == LBM_D2Q5 ? 5 : 9);
    int rc = LBM_OK;
    // the populations and the production field of the current level, and its phi (ghost layers included: they are images of nodes)
    if (c->L.es == 8) {
        rc = count_array<double>(c, c->L.off_f[c->cur], qf * N, counter);
        if (!rc) rc = count_array<double>(c, c->L.off_g[c->cur], qg * N, counter);
        if (!rc) rc = count_array<double>(c, c->L.off_s[c->cur], qs * N, counter);
        if (!rc) rc = count_array<double>(c, c->L.off_pdot[c->cur], N, counter);
    } else {
        rc = count_array<float>(c, c->L.off_f[c->cur], qf * N, counter);
        if (!rc) rc = count_array<float>(c, c->L.off_g[c->cur], qg * N, counter);
        if (!rc) rc = count_array<float>(c, c->L.off_s[c->cur], qs * N, counter);
        if (!rc) rc = count_array<float>(c, c->L.off_pdot[c->cur], N, counter);
    }
    if (!rc) rc = count_array<double>(c, c->L.off_phi[c->curphi], c->L.phi_pad_elems, counter);
    if (rc) return rc;
    unsigned long long h = 0;
    CK(cudaMemcpyAsync(&h, counter, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    *n_bad = (long long)h;
    return LBM_OK;
}
