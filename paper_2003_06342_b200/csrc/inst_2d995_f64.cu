// Instantiation unit: (D2Q9, D2Q9, D2Q5) in double.  One translation unit per (lattice set, precision) so that the build
// compiles them in parallel.
#include "impl.cuh"

namespace lbm {
const ImplOps *ops_2d995_f64(int nx) {
    if (wide_tile_pays(nx)) return Impl<D2Q9, D2Q9, D2Q5, double, TileWide2K>::ops();
    return Impl<D2Q9, D2Q9, D2Q5, double, TileNarrow2>::ops();
}
}  // namespace lbm
