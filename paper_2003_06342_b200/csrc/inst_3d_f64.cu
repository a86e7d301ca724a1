// Instantiation unit: (D3Q19, D3Q7, D3Q7) in double.  One translation unit per (lattice set, precision) so that the build
// compiles them in parallel.
#include "impl.cuh"

namespace lbm {
const ImplOps *ops_3d_f64(int nx) {
    if (wide_tile_pays(nx)) return Impl<D3Q19, D3Q7, D3Q7, double, TileWide3>::ops();
    if (nx >= 64 && nx % 64 == 0) return Impl<D3Q19, D3Q7, D3Q7, double, TileMid3>::ops();
    return Impl<D3Q19, D3Q7, D3Q7, double, TileNarrow3>::ops();
}
}  // namespace lbm
