// Lattice tables of the CUDA path.  Compile-time tables: every loop over directions is fully
// unrolled, so e_i, w_i and the opposite index fold into immediates and per-direction code.
// D2Q9 weights are the standard ones, D2Q5 is not in the paper (reading S1).
// Direction order: D2Q9 as printed in the paper; 3D: e1..6 = +x,+y,+z,-x,-y,-z, then the
// pairs the paper prints for D3Q19 / the cube diagonals of D3Q15.
#pragma once

namespace lbm {

struct D2Q5 {
    static constexpr int Q = 5;
    static constexpr int D = 2;
    static constexpr double e2 = 1.0 / 3.0;
    __host__ __device__ static constexpr int ex(int i) { constexpr int t[Q] = {0, 1, 0, -1, 0}; return t[i]; }
    __host__ __device__ static constexpr int ey(int i) { constexpr int t[Q] = {0, 0, 1, 0, -1}; return t[i]; }
    __host__ __device__ static constexpr int ez(int) { return 0; }
    __host__ __device__ static constexpr int opp(int i) { constexpr int t[Q] = {0, 3, 4, 1, 2}; return t[i]; }
    __host__ __device__ static constexpr double w(int i) { return i == 0 ? 1.0 / 3.0 : 1.0 / 6.0; }
};

struct D2Q9 {
    static constexpr int Q = 9;
    static constexpr int D = 2;
    static constexpr double e2 = 1.0 / 3.0;
    __host__ __device__ static constexpr int ex(int i) { constexpr int t[Q] = {0, 1, 0, -1, 0, 1, -1, -1, 1}; return t[i]; }
    __host__ __device__ static constexpr int ey(int i) { constexpr int t[Q] = {0, 0, 1, 0, -1, 1, 1, -1, -1}; return t[i]; }
    __host__ __device__ static constexpr int ez(int) { return 0; }
    __host__ __device__ static constexpr int opp(int i) { constexpr int t[Q] = {0, 3, 4, 1, 2, 7, 8, 5, 6}; return t[i]; }
    __host__ __device__ static constexpr double w(int i) { return i == 0 ? 4.0 / 9.0 : (i < 5 ? 1.0 / 9.0 : 1.0 / 36.0); }
};

struct D3Q7 {
    static constexpr int Q = 7;
    static constexpr int D = 3;
    static constexpr double e2 = 1.0 / 4.0;
    __host__ __device__ static constexpr int ex(int i) { constexpr int t[Q] = {0, 1, 0, 0, -1, 0, 0}; return t[i]; }
    __host__ __device__ static constexpr int ey(int i) { constexpr int t[Q] = {0, 0, 1, 0, 0, -1, 0}; return t[i]; }
    __host__ __device__ static constexpr int ez(int i) { constexpr int t[Q] = {0, 0, 0, 1, 0, 0, -1}; return t[i]; }
    __host__ __device__ static constexpr int opp(int i) { constexpr int t[Q] = {0, 4, 5, 6, 1, 2, 3}; return t[i]; }
    __host__ __device__ static constexpr double w(int i) { return i == 0 ? 1.0 / 4.0 : 1.0 / 8.0; }
};

struct D3Q19 {
    static constexpr int Q = 19;
    static constexpr int D = 3;
    static constexpr double e2 = 1.0 / 3.0;
    __host__ __device__ static constexpr int ex(int i) {
        constexpr int t[Q] = {0, 1, 0, 0, -1, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
        return t[i];
    }
    __host__ __device__ static constexpr int ey(int i) {
        constexpr int t[Q] = {0, 0, 1, 0, 0, -1, 0, 1, 1, -1, -1, 0, 0, 0, 0, 1, -1, 1, -1};
        return t[i];
    }
    __host__ __device__ static constexpr int ez(int i) {
        constexpr int t[Q] = {0, 0, 0, 1, 0, 0, -1, 0, 0, 0, 0, 1, 1, -1, -1, 1, 1, -1, -1};
        return t[i];
    }
    __host__ __device__ static constexpr int opp(int i) {
        constexpr int t[Q] = {0, 4, 5, 6, 1, 2, 3, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};
        return t[i];
    }
    __host__ __device__ static constexpr double w(int i) { return i == 0 ? 1.0 / 3.0 : (i < 7 ? 1.0 / 18.0 : 1.0 / 36.0); }
};

// PAPER.md:190 prints e7 = (1,1,1), e8 = (-1,1,1), ..., e14 = (1,-1,-1); the elided vectors go counter-clockwise around z
// on each level (reading G10).
struct D3Q15 {
    static constexpr int Q = 15;
    static constexpr int D = 3;
    static constexpr double e2 = 1.0 / 3.0;
    __host__ __device__ static constexpr int ex(int i) {
        constexpr int t[Q] = {0, 1, 0, 0, -1, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
        return t[i];
    }
    __host__ __device__ static constexpr int ey(int i) {
        constexpr int t[Q] = {0, 0, 1, 0, 0, -1, 0, 1, 1, -1, -1, 1, 1, -1, -1};
        return t[i];
    }
    __host__ __device__ static constexpr int ez(int i) {
        constexpr int t[Q] = {0, 0, 0, 1, 0, 0, -1, 1, 1, 1, 1, -1, -1, -1, -1};
        return t[i];
    }
    __host__ __device__ static constexpr int opp(int i) {
        constexpr int t[Q] = {0, 4, 5, 6, 1, 2, 3, 13, 14, 11, 12, 9, 10, 7, 8};
        return t[i];
    }
    __host__ __device__ static constexpr double w(int i) { return i == 0 ? 2.0 / 9.0 : (i < 7 ? 1.0 / 9.0 : 1.0 / 72.0); }
};

// compile-time self-check: opp(i) really is the direction -e_i
template <class L> constexpr bool lattice_consistent() {
    for (int i = 0; i < L::Q; ++i) {
        int j = L::opp(i);
        if (L::ex(j) != -L::ex(i) || L::ey(j) != -L::ey(i) || L::ez(j) != -L::ez(i)) return false;
    }
    return true;
}
static_assert(lattice_consistent<D2Q5>() && lattice_consistent<D2Q9>() && lattice_consistent<D3Q7>() &&
              lattice_consistent<D3Q19>() && lattice_consistent<D3Q15>(), "opposite table broken");

}  // namespace lbm
