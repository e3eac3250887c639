// homg_geom.h — geometry of one level array, shared by host code and kernels.
#pragma once

namespace homg {

struct LevelGeom {
    int nx, ny, nz;      // nodes per axis incl. boundary (nz = 1 in 2-D)
    int px;              // row pitch in elements
    long long pp;        // plane pitch in elements (px*ny)
};

// Variable-coefficient stencil (R11): harmonic-mean face coefficients, precomputed per level at
// homg_set_coefficient (S0).  z[c] / y[c] / x[c] = 2 k_c k_q / (k_c + k_q) for the face between node c and
// its +z / +y / +x neighbour q (0 where q does not exist).  The face value is symmetric in (c, q), so
// both nodes of a face read the very number the oracle computes from either side.
template <class T>
struct Faces {
    const T* z;
    const T* y;
    const T* x;
};

template <class T>
struct Coef {            // per-level operator constants
    T ih2;               // 1/h_m^2
    T w;                 // omega
    T w_over_D;          // omega / (2d/h_m^2)      (constant coefficient)
    T twod;              // 2d
    T D;                 // 2d * (1/h_m^2), rounded as the kernels round it (constant coefficient)
    T rD;                // RN(1/D)
    T h2;                // h_m^2                     (Eq. 3 form of the constant-coefficient sweep)
    T wp;                // omega / 2d
};

}  // namespace homg
