// hydro_faces.cuh -- per-direction building blocks shared by the stage kernels: limited face values
// of one cell, HLL flux through a face of given normal, primitives of one cell.  The production build
// takes them from hydro_math_fast.cuh, the verification build (-DHYDRO_VERIFY, -fmad=false) from
// hydro_math.cuh (the oracle's association, operation for operation).
#pragma once
#include "hydro_math.cuh"
#ifndef HYDRO_VERIFY
#include "hydro_math_fast.cuh"
#endif

namespace hyd {

// ---- per-direction helpers: primitives are always held as (rho, vx, vy, vz, p) -----------------

// slope of one cell from its two neighbours along a direction; returns inner and outer values
__device__ __forceinline__ void limited_faces(double theta, const double Wm[5], const double Wc[5],
                                              const double Wp[5], double inner[5], double outer[5])
{
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double a = Wc[v] - Wm[v];
        const double b = Wp[v] - Wc[v];
        const double s = minmod(theta, a, b);
        inner[v] = Wc[v] - 0.5 * s;
        outer[v] = Wc[v] + 0.5 * s;
    }
}
#ifndef HYDRO_VERIFY
#define HYD_LIMITED_FACES(theta, Wm, Wc, Wp, In, Ou) fast::limited_faces(0.5 * (theta), Wm, Wc, Wp, In, Ou)
#define HYD_HLL fast::hll_flux
#define HYD_PRIM5 fast::prim5
#define HYD_SUM3(x, y, z) (((x) + (y)) + (z))
#else
#define HYD_LIMITED_FACES(theta, Wm, Wc, Wp, In, Ou) limited_faces(theta, Wm, Wc, Wp, In, Ou)
#define HYD_HLL hll_flux
#define HYD_PRIM5 prim5
#define HYD_SUM3(x, y, z) sum3(x, y, z)
#endif

// HLL flux through a face with normal D; L, R in (rho,vx,vy,vz,p); F in (rho,mx,my,mz,E) order
template <int D>
__device__ __forceinline__ void face_flux(const double L[5], const double R[5], double gamma,
                                          double igm1, double F[5])
{
    const double l[5] = { L[0], L[1 + D], L[1 + (D + 1) % 3], L[1 + (D + 2) % 3], L[4] };
    const double r[5] = { R[0], R[1 + D], R[1 + (D + 1) % 3], R[1 + (D + 2) % 3], R[4] };
    double f[5];
    HYD_HLL(l, r, gamma, igm1, f);
    F[0] = f[0];
    F[1 + D] = f[1];
    F[1 + (D + 1) % 3] = f[2];
    F[1 + (D + 2) % 3] = f[3];
    F[4] = f[4];
}

__device__ __forceinline__ void prim5(const double U[5], double gm1, double W[5])
{
    const Prim w = primitive(U[0], U[1], U[2], U[3], U[4], gm1);
    W[0] = w.rho; W[1] = w.vx; W[2] = w.vy; W[3] = w.vz; W[4] = w.p;
}

}  // namespace hyd
