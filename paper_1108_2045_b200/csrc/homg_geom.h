// homg_geom.h — geometry of one level array, shared by host code and kernels.
#pragma once

namespace homg {

struct LevelGeom {
    int nx, ny, nz;      // nodes per axis incl. boundary (nz = 1 in 2-D)
    int px;              // row pitch in elements
    long long pp;        // plane pitch in elements (px*ny)
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
