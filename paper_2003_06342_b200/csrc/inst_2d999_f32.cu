// Instantiation unit: (D2Q9, D2Q9, D2Q9) in float, phi kept in double (include/lbm.h "precision").  One translation unit per
// (lattice set, precision) so that the build compiles them in parallel.
#include "impl.cuh"

namespace lbm {
const ImplOps *ops_2d999_f32(int nx) {
    if (wide_tile_pays(nx)) return Impl<D2Q9, D2Q9, D2Q9, float, TileWide2K, float, double>::ops();
    return Impl<D2Q9, D2Q9, D2Q9, float, TileNarrow2, float, double>::ops();
}
}  // namespace lbm
