// Instantiation unit: (D3Q15, D3Q7, D3Q7) in float, phi kept in double (include/lbm.h "precision").  One translation unit per
// (lattice set, precision) so that the build compiles them in parallel.
#include "impl.cuh"

namespace lbm {
const ImplOps *ops_3d15_f32(int nx) {
    if (wide_tile_pays(nx)) return Impl<D3Q15, D3Q7, D3Q7, float, TileWide3Phi, float, double>::ops();
    if (nx >= 64 && nx % 64 == 0) return Impl<D3Q15, D3Q7, D3Q7, float, TileMid3Phi, float, double>::ops();   // 64 x 4: 128 threads of pairs
    return Impl<D3Q15, D3Q7, D3Q7, float, TileNarrow3, float, double>::ops();
}
}  // namespace lbm
