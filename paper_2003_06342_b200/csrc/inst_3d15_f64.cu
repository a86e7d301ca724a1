// Instantiation unit: (D3Q15, D3Q7, D3Q7) in double -- the paper's other 3D Navier-Stokes lattice.
#include "impl.cuh"

namespace lbm {
const ImplOps *ops_3d15_f64(int nx) {
    if (wide_tile_pays(nx)) return Impl<D3Q15, D3Q7, D3Q7, double, TileWide3>::ops();
    if (nx >= 64 && nx % 64 == 0) return Impl<D3Q15, D3Q7, D3Q7, double, TileMid3>::ops();
    return Impl<D3Q15, D3Q7, D3Q7, double, TileNarrow3>::ops();
}
}  // namespace lbm
