// hydro_math.cuh -- per-cell / per-face arithmetic of the RK2 Euler step, device side.
//
// Written from DESIGN.md section 3 (steps O2-O7, readings R1-R20); shares nothing with oracle/.
// The association of every expression below is part of the definition: compiled with
// -fmad=false (verification build) it reproduces the oracle's roundings one for one; compiled
// with -fmad=true (production build) ptxas contracts a*b+c into DFMA and results differ at
// roundoff (R20).
#pragma once
#include <cuda_runtime.h>

namespace hyd {

constexpr int NVAR = 5;   // rho, m_x, m_y, m_z, E  |  rho, v_x, v_y, v_z, p
constexpr int NG = 2;     // ghost layers per side

// explicit comparisons: the same NaN / signed-zero behaviour on every build
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

// R17: permutation-symmetric three-term sum = (smallest + largest) + middle.
__device__ __forceinline__ double sum3(double a, double b, double c)
{
    const double lo = dmin(a, b), hi = dmax(a, b);
    const double s0 = dmin(lo, c), s2 = dmax(hi, c);
    const double s1 = dmax(lo, dmin(hi, c));
    return (s0 + s2) + s1;
}

// O3 / R4: generalized minmod of the backward difference a and forward difference b.
__device__ __forceinline__ double minmod(double theta, double a, double b)
{
    const double ta = theta * fabs(a);
    const double tb = theta * fabs(b);
    const double tc = 0.5 * fabs(a + b);
    const double m = dmin(dmin(ta, tb), tc);
    double s = 0.0;
    if (a > 0.0 && b > 0.0) s = m;
    if (a < 0.0 && b < 0.0) s = -m;
    return s;
}

struct Prim { double rho, vx, vy, vz, p; };

// O2: conserved -> primitive.  `inv` (1/rho) and `q` (|v|^2) are returned for the CFL epilogue.
__device__ __forceinline__ Prim primitive(double rho, double mx, double my, double mz, double E,
                                          double gm1, double &inv, double &q)
{
    Prim w;
    inv = 1.0 / rho;
    w.rho = rho;
    w.vx = mx * inv; w.vy = my * inv; w.vz = mz * inv;
    q = sum3(w.vx * w.vx, w.vy * w.vy, w.vz * w.vz);
    const double hr = 0.5 * rho;
    const double ke = hr * q;
    const double ei = E - ke;
    w.p = gm1 * ei;
    return w;
}

__device__ __forceinline__ Prim primitive(double rho, double mx, double my, double mz, double E,
                                          double gm1)
{
    double inv, q;
    return primitive(rho, mx, my, mz, E, gm1, inv, q);
}

// O7: signal speed |v| + c_s of a cell, from O2's by-products.
__device__ __forceinline__ double signal_speed(const Prim &w, double inv, double q, double gamma)
{
    const double gp = gamma * w.p;
    const double c2 = gp * inv;
    return sqrt(q) + sqrt(c2);
}

// One side of a face (O4).  Velocities are passed as (normal, t1, t2) = cyclic order starting at
// the face axis, so the three directions run the same code.
struct Side { double U[5]; double F[5]; double vn, c; };   // component order: rho, n, t1, t2, E

__device__ __forceinline__ void side_state(double rho, double vn, double vt1, double vt2, double p,
                                           double gamma, double igm1, Side &s)
{
    const double gp = gamma * p;
    const double c2 = gp / rho;
    s.c = sqrt(c2);
    const double tt = vt1 * vt1 + vt2 * vt2;
    const double k = vn * vn + tt;
    const double hr = 0.5 * rho;
    const double E = p * igm1 + hr * k;
    s.U[0] = rho; s.U[1] = rho * vn; s.U[2] = rho * vt1; s.U[3] = rho * vt2; s.U[4] = E;
    s.F[0] = s.U[1];
    s.F[1] = s.U[1] * vn + p;
    s.F[2] = s.U[2] * vn;
    s.F[3] = s.U[3] * vn;
    s.F[4] = (E + p) * vn;
    s.vn = vn;
}

// O4 / R6: HLL flux, components in (rho, n, t1, t2, E) order.
__device__ __forceinline__ void hll_flux(const double L[5], const double R[5], double gamma,
                                         double igm1, double F[5])
{
    Side sl, sr;
    side_state(L[0], L[1], L[2], L[3], L[4], gamma, igm1, sl);
    side_state(R[0], R[1], R[2], R[3], R[4], gamma, igm1, sr);
    const double ap = dmax(0.0, dmax(sl.vn + sl.c, sr.vn + sr.c));
    const double am = dmax(0.0, dmax(sl.c - sl.vn, sr.c - sr.vn));
    const double w = 1.0 / (ap + am);
    const double pi = ap * am;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double num = (ap * sl.F[v] + am * sr.F[v]) - pi * (sr.U[v] - sl.U[v]);
        F[v] = __dmul_rn(num, w);   // never contracted into a consumer's subtract: equal
                                    // face states must give bit-equal fluxes on every build (P1)
    }
}

}  // namespace hyd
