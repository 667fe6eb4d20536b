// hydro_math_fast.cuh -- production-build arithmetic of the fused stage kernel.
//
// Same formulas as hydro_math.cuh (O2-O7) with the freedoms the production
// build takes (R20 and section 6): FMA contraction, branch-free reciprocal / reciprocal
// square root built on MUFU.RCP64H / MUFU.RSQ64H seeds plus Newton steps (<= 2 ulp instead of
// correctly rounded), sign handling of the limiter on the integer pipe, plain (x+y)+z instead of
// the sorted three-term sum.  Results differ from the oracle at roundoff only; the parity bar for
// this build is relL1 <= 1e-10, relLinf <= 1e-8 (BASELINE.json:north_star).  The verification
// build (-DHYDRO_VERIFY, -fmad=false) never includes this path.
//
// Why: the fp64 pipe and the issue slots are two of the three units the stage kernel keeps about half
// busy (the third is the shared-memory crossbar), so
// every DSETP/FSEL pair and every slow-path branch of the IEEE divide / sqrt costs throughput.
#pragma once
#include "hydro_math.cuh"

namespace hyd {
namespace fast {

// 1/x, x > 0 finite and normal.  The MUFU.RCP64H seed is good to ~2^-20; one third-order step
// y (1 + e + e^2), e = 1 - x y, leaves e^3 ~ 2^-60 plus the rounding of the last fma (<= 1 ulp
// measured; the previous form, two Newton steps, cost one more DFMA).
__device__ __forceinline__ double rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

// 1/sqrt(x), x > 0 finite and normal.  One third-order step on the ~2^-20 seed: measured on
// B200 |x y^2 - 1| <= 1.3 eps over 2^26 arguments (a second step does not improve on that).
__device__ __forceinline__ double rsqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y * y, 1.0);           // 1 - x y^2
    const double p = fma(0.375, e, 0.5);
    return fma(y, p * e, y);                        // y (1 + e/2 + 3 e^2/8)
}

// min of two non-negative doubles on the integer pipe (DSETP runs at half the DFMA rate on
// sm_100a, measured; non-negative doubles order like their bit patterns)
__device__ __forceinline__ double min_nonneg(double x, double y)
{
    return __double_as_longlong(x) < __double_as_longlong(y) ? x : y;
}

__device__ __forceinline__ double max_nonneg(double x, double y)
{
    return __double_as_longlong(x) > __double_as_longlong(y) ? x : y;
}

// max(0, x) on the sign bit: one integer max on the high word.  A negative x keeps its low word, i.e.
// comes back as a denormal below 2^-1022 instead of 0 -- far below the roundoff of every sum it enters
// (it only feeds a+ + a- and the HLL weights), and two instructions cheaper than clearing it.
__device__ __forceinline__ double max0(double x)
{
    return __hiloint2double(max(__double2hiint(x), 0), __double2loint(x));
}

// O2: conserved -> primitive (rho, vx, vy, vz, p)
__device__ __forceinline__ void prim5(const double U[5], double gm1, double W[5])
{
    const double inv = rcp(U[0]);
    W[0] = U[0];
    W[1] = U[1] * inv; W[2] = U[2] * inv; W[3] = U[3] * inv;
    const double rq = fma(U[1], W[1], fma(U[2], W[2], U[3] * W[3]));     // rho |v|^2 = m . v
    W[4] = gm1 * fma(-0.5, rq, U[4]);
}

// O3: limited slope of one cell, hs = 0.5 * sigma, in a select-free form on the fp64 pipe (the
// kernel is limited by issue slots as much as by the pipe; the comparison form costs 11 integer /
// select instructions per slope, this one a single LOP3).  With c = a + b = W(+1) - W(-1) and
// d = a - b:
//   g = |c| - |d| = +2 min(|a|,|b|) when a and b agree in sign, -2 min(|a|,|b|) otherwise;
//   T = theta|g| + |c| - |theta g - |c|| = 2 clamp(theta g, 0, |c|)      (clamp(x,0,y) = (|x| + y - |x-y|)/2)
//     = 4 min(theta|a|, theta|b|, |a+b|/2) when the signs agree, exactly 0 otherwise;
//   hs = T/8 with the sign of c.
// Exact where it matters (a = b = 0 gives 0; opposite signs give exactly 0); elsewhere within a
// few ulp of the jump |c| of the comparison form (R20).  Nine fp64 instructions.
__device__ __forceinline__ void limited_faces(double half_theta, const double Wm[5],
                                              const double Wc[5], const double Wp[5],
                                              double inner[5], double outer[5])
{
    const double th = 2.0 * half_theta;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double c = Wp[v] - Wm[v];
        const double d = fma(2.0, Wc[v], -Wm[v]) - Wp[v];
        const double g = fabs(c) - fabs(d);
        const double u = fma(th, g, -fabs(c));
        const double w = fma(th, fabs(g), fabs(c));
        const double T = w - fabs(u);
        const double Ts = __hiloint2double(__double2hiint(T) | (__double2hiint(c) & 0x80000000), __double2loint(T));
        inner[v] = fma(-0.125, Ts, Wc[v]);
        outer[v] = fma(0.125, Ts, Wc[v]);
    }
}

// O4: HLL flux, components in (rho, n, t1, t2, E) order; inputs (rho, vn, vt1, vt2, p).
// With F_S = U_S vn_S + P_S, P = (0, p, 0, 0, p vn), the HLL combination
//     [a+ F_L + a- F_R - a+ a- (U_R - U_L)] / (a+ + a-)
// is regrouped per side as  alpha (U_L (vn_L + a-) + P_L) + beta (U_R (vn_R - a+) + P_R),  alpha = a+ w,
// beta = a- w:  neither the physical fluxes nor the jump U_R - U_L are formed, the momenta appear only
// through rho (vn +- a) and the sound speed only inside the wave-speed fmas -- 60 fp64 instructions per
// face instead of 75.  Same value up to roundoff (R20); the two sides' terms of size
// rho c / 2 cancel where the classical form subtracts nearly equal states, so the absolute error per
// face is eps rho c instead of eps |U_R - U_L| c: still at the rounding level of the state itself.
__device__ __forceinline__ void hll_flux(const double L[5], const double R[5], double gamma,
                                         double igm1, double F[5])
{
    const double gpL = gamma * L[4], gpR = gamma * R[4];
    const double rsL = rsqrt(gpL * L[0]), rsR = rsqrt(gpR * R[0]);       // c = gp rs
    const double ap = max0(dmax(fma(gpL, rsL, L[1]), fma(gpR, rsR, R[1])));
    const double am = max0(dmax(fma(gpL, rsL, -L[1]), fma(gpR, rsR, -R[1])));
    const double w = rcp(ap + am);
    const double al = ap * w, be = am * w;
    double XL[5], XR[5];
    {
        const double s = L[1] + am;
        const double q = fma(L[1], L[1], fma(L[2], L[2], L[3] * L[3]));
        const double E = fma(0.5 * L[0], q, L[4] * igm1);
        XL[0] = L[0] * s; XL[1] = fma(XL[0], L[1], L[4]); XL[2] = XL[0] * L[2]; XL[3] = XL[0] * L[3];
        XL[4] = fma(E, s, L[4] * L[1]);
    }
    {
        const double s = R[1] - ap;
        const double q = fma(R[1], R[1], fma(R[2], R[2], R[3] * R[3]));
        const double E = fma(0.5 * R[0], q, R[4] * igm1);
        XR[0] = R[0] * s; XR[1] = fma(XR[0], R[1], R[4]); XR[2] = XR[0] * R[2]; XR[3] = XR[0] * R[3];
        XR[4] = fma(E, s, R[4] * R[1]);
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) F[v] = fma(al, XL[v], be * XR[v]);
}

// O7: signal speed |v| + c_s of one updated cell for the fused CFL reduction.  sqrt(x) is formed as
// x * rsqrt(x + tiny) so that x = 0 gives 0 instead of NaN.  `bad` is raised on the sign/zero bits
// of rho and p (integer pipe); a non-finite speed is caught once per thread from the running
// maximum, whose bit pattern then compares above every finite value.
__device__ __forceinline__ double signal_speed(const double U[5], double gamma, double gm1, int &bad)
{
    double W[5];
    const double inv = rcp(U[0]);
    W[1] = U[1] * inv; W[2] = U[2] * inv; W[3] = U[3] * inv;
    const double q = fma(W[1], W[1], fma(W[2], W[2], W[3] * W[3]));
    const double p = gm1 * fma(-0.5 * U[0], q, U[4]);
    const double c2 = (gamma * p) * inv;
    const double tiny = 1e-300;
    const double s = fma(q, rsqrt(q + tiny), c2 * rsqrt(c2 + tiny));
    bad |= (__double_as_longlong(U[0]) <= 0ll) | (__double_as_longlong(p) <= 0ll);
    return s;
}

}  // namespace fast
}  // namespace hyd
