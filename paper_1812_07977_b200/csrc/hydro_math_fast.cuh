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
// Why: the stage kernel is bound by the fp64 pipe and by issue slots, so
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
__device__ __forceinline__ void hll_flux(const double L[5], const double R[5], double gamma,
                                         double igm1, double F[5])
{
    double UL[5], UR[5], FL[5], FR[5], cL, cR;
    {
        const double gp = gamma * L[4];
        cL = gp * rsqrt(gp * L[0]);
        UL[0] = L[0]; UL[1] = L[0] * L[1]; UL[2] = L[0] * L[2]; UL[3] = L[0] * L[3];
        const double rk = fma(UL[1], L[1], fma(UL[2], L[2], UL[3] * L[3]));     // rho |v|^2
        const double E = fma(0.5, rk, L[4] * igm1);
        UL[4] = E;
        FL[0] = UL[1]; FL[1] = fma(UL[1], L[1], L[4]); FL[2] = UL[2] * L[1]; FL[3] = UL[3] * L[1];
        FL[4] = (E + L[4]) * L[1];
    }
    {
        const double gp = gamma * R[4];
        cR = gp * rsqrt(gp * R[0]);
        UR[0] = R[0]; UR[1] = R[0] * R[1]; UR[2] = R[0] * R[2]; UR[3] = R[0] * R[3];
        const double rk = fma(UR[1], R[1], fma(UR[2], R[2], UR[3] * R[3]));
        const double E = fma(0.5, rk, R[4] * igm1);
        UR[4] = E;
        FR[0] = UR[1]; FR[1] = fma(UR[1], R[1], R[4]); FR[2] = UR[2] * R[1]; FR[3] = UR[3] * R[1];
        FR[4] = (E + R[4]) * R[1];
    }
    const double ap = max0(dmax(L[1] + cL, R[1] + cR));
    const double am = max0(dmax(cL - L[1], cR - R[1]));
    const double w = rcp(ap + am);
    const double al = ap * w, be = am * w, de = al * am;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double f = fma(al, FL[v], be * FR[v]);
        F[v] = __fma_rn(-de, UR[v] - UL[v], f);
    }
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
