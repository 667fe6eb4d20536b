// hydro_stage_warp2d.cuh -- "warp column" RK-stage kernel of 2D runs (R21).
//
// The 3D kernel's idea -- march along the last active axis with a register pipeline so that nothing in
// that direction is recomputed or exchanged -- applied to two dimensions leaves only ONE lateral
// direction, x, and 32 cells of x are one warp.  So here a warp is the whole unit of work: it owns a
// strip of the row 32 lanes wide and marches down y; the y direction lives in its registers (W(j-2),
// W(j-1), the outer y-face value and the last y-flux), the x direction is exchanged with warp shuffles
// (primitives of the x-neighbours, the outer face value to lane+1, the flux back to lane-1).  No shared
// memory, no barriers, no block-wide phases: every warp is independent, 16 of them per SM.
//
// Lanes 0, 1, 30, 31 of a strip are halo cells (their slopes feed the faces of lanes 2 and 29); the 28
// lanes between own the cells that are updated, so strips advance by 28 cells and one eighth of the
// slopes / fluxes is redundant -- the price of having no special lanes and no divergence.  The boundary
// rule of both axes is applied on the way in: a lane whose cell is a ghost cell, and a row that is a
// ghost row, read their source cell / row (clamp, mirror with the normal momentum negated, wrap), so no
// ghost layer in memory is ever read or written (no ghost fill, no wrap stores: three launches per step
// for every boundary mix).  The own conserved values are read again from L1 / L2 when their row is
// completed two rows later.  Same building blocks as the other stage kernels (hydro_faces.cuh): the
// verification build reproduces the oracle bit for bit.
#pragma once
#include "hydro_kernels.cuh"

namespace hyd {

constexpr int W2_OWN = 28;             // cells updated per strip (lanes 2 .. 29)
constexpr int W2_WARPS = 4;            // warps per block (independent of one another)

struct Warp2dArgs {
    Grid g;
    const double *Uin;
    const double *Uold;     // stage 2: U0 (own cell only); may alias Uout
    double *Uout;
    double dt_over_dx;      // used when dev_dt == nullptr
    const StepScalars *dev_dt;
    double dx;
    StepScalars *red;       // stage 2: max-signal-speed accumulator + sticky flag (or nullptr)
    int nstrip, nchunk, rows;   // strips along x, chunks along y of `rows` rows each
};

template <int STAGE, bool ANISO>
__global__ void __launch_bounds__(32 * W2_WARPS, 4)
stage_warp2d_kernel(const Warp2dArgs a)
{
    const Grid &g = a.g;
    const int lane = threadIdx.x & 31;
    const int item = blockIdx.x * W2_WARPS + (threadIdx.x >> 5);       // (strip, chunk), strip fastest
    double smax = 0.0;
    int bad = 0;
    if (item < a.nstrip * a.nchunk) {
        const int chunk = item / a.nstrip, strip = item - chunk * a.nstrip;
        const int j0 = chunk * a.rows, nc = min(a.rows, g.ny - j0);    // rows [j0, j0 + nc)
        const int i = strip * W2_OWN - NG + lane;                       // this lane's cell (may be a ghost cell)
        const bool owner = lane >= NG && lane < NG + W2_OWN && i < g.nx;
        const double gamma = g.gamma, gm1 = g.gm1, igm1 = g.igm1, theta = g.theta;
        const double r = a.dev_dt ? a.dev_dt->dt / a.dx : a.dt_over_dx;
        const long long sv = g.sv;
        bool fx = false;
        const int is = bc_source(i, g.nx, g.bc[0], g.bc[1], 0, g.nx - 1, fx);
        const long long cx = cell0(g, is, 0, 0);                        // source column of this lane
        // primitives of this lane's cell in row jj (a ghost row reads its source row)
        auto load_row = [&](int jj, double W[5]) {
            bool fy = false;
            const int js = bc_source(jj, g.ny, g.bc[2], g.bc[3], 0, g.ny - 1, fy);
            const long long c = cx + (long long)g.px * js;
            double U[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) U[v] = __ldg(a.Uin + v * sv + c);
            U[1] = flip_sign(U[1], fx); U[2] = flip_sign(U[2], fy);
            HYD_PRIM5(U, gm1, W);
        };

        // ---- prologue: rows j0-2 .. j0+1 -> W(j0), W(j0+1), outer_y(j0), flux through face j0-1/2 ----
        double Wa[5], Wb[5], Oy[5], Fym[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) { Wa[v] = Wb[v] = Oy[v] = Fym[v] = 0.0; }
#pragma unroll 1
        for (int p = 0; p < 4; ++p) {
            double Wn[5];
            load_row(j0 - NG + p, Wn);
            if (p >= 2) {
                double Iy[5], Oyn[5];
                HYD_LIMITED_FACES(theta, Wa, Wb, Wn, Iy, Oyn);           // cell of row j0-2+p-1
                if (p == 3) face_flux<1>(Oy, Iy, gamma, igm1, Fym);
#pragma unroll
                for (int v = 0; v < 5; ++v) Oy[v] = Oyn[v];
            }
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wa[v] = Wb[v]; Wb[v] = Wn[v]; }
        }

#pragma unroll 1
        for (int c = 0; c < nc; ++c) {
            const int j = j0 + c;
            const long long cg = cell0(g, i < g.nx ? max(i, 0) : g.nx - 1, j, 0);   // own cell (owners: i in range)
            // own conserved values of row j (L1 / L2; stage 2's U0 from DRAM), in flight while the x direction
            // is computed
            double u1[5], u0[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                u1[v] = __ldg(a.Uin + v * sv + cg);
                if (STAGE == 2) u0[v] = owner ? a.Uold[v * sv + cg] : 0.0;      // (in place: only the owner may look)
            }
            // ---- x direction of row j (W = Wa): neighbours, outer value and flux through the warp ----
            double Fxl[5], dFx[5];
            {
                double Wm[5], Wp[5], Ix[5], Ox[5], L[5];
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    Wm[v] = __shfl_up_sync(0xffffffffu, Wa[v], 1);
                    Wp[v] = __shfl_down_sync(0xffffffffu, Wa[v], 1);
                }
                HYD_LIMITED_FACES(theta, Wm, Wa, Wp, Ix, Ox);            // valid on lanes 1 .. 30
#pragma unroll
                for (int v = 0; v < 5; ++v) L[v] = __shfl_up_sync(0xffffffffu, Ox[v], 1);
                face_flux<0>(L, Ix, gamma, igm1, Fxl);                   // low face: valid on lanes 2 .. 30
#pragma unroll
                for (int v = 0; v < 5; ++v) dFx[v] = __shfl_down_sync(0xffffffffu, Fxl[v], 1) - Fxl[v];
            }
            // ---- y direction: primitives of row j+2, slope of row j+1, flux through face j+1/2 ----
            double Wn[5], Iy[5], Oyn[5], Fyp[5];
            load_row(j + NG, Wn);
            HYD_LIMITED_FACES(theta, Wa, Wb, Wn, Iy, Oyn);
            face_flux<1>(Oy, Iy, gamma, igm1, Fyp);
            // ---- update of row j ----
            double un[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                double dFy = Fyp[v] - Fym[v];
                if (ANISO) dFy = g.ry * dFy;                             // non-cubic cells (R23): dx/dy
                const double D = dFx[v] + dFy;
                const double dU = -(r * D);
                if (STAGE == 1) {
                    un[v] = u1[v] + dU;
                } else {
                    const double sum = u0[v] + u1[v];
                    un[v] = 0.5 * (sum + dU);
                }
                Fym[v] = Fyp[v]; Oy[v] = Oyn[v]; Wa[v] = Wb[v]; Wb[v] = Wn[v];
            }
            if (owner) {
#pragma unroll
                for (int v = 0; v < 5; ++v) a.Uout[v * sv + cg] = un[v];
                if (STAGE == 2 && a.red) {
#ifdef HYDRO_VERIFY
                    const double s = cell_signal_speed(un[0], un[1], un[2], un[3], un[4], gamma, gm1, bad);
                    smax = s > smax ? s : smax;
#else
                    smax = fast::max_nonneg(smax, fast::signal_speed(un, gamma, gm1, bad));
#endif
                }
            }
        }
    }
    if (STAGE == 2 && a.red) {
        if (!(smax <= 1.79769313486231570e308)) { bad = 1; smax = 0.0; }   // inf or NaN pattern won
        block_max_to_global(smax, bad, &a.red->smax_bits, &a.red->flag);
    }
}

// Rows per chunk: the (strip, chunk) items should fill whole waves of the resident warps (16 per SM); a
// chunk of l rows costs about l + 3 row times (four warm-up rows of primitives and y-slopes).
inline int warp2d_choose_rows(const Grid &g, int nsm)
{
    const long long nstrip = (g.nx + W2_OWN - 1) / W2_OWN, slots = (long long)nsm * 16;
    int best = g.ny;
    double best_cost = 1e300;
    for (int nch = 1; nch <= (g.ny + 7) / 8; ++nch) {
        const int rows = (g.ny + nch - 1) / nch;
        const long long items = nstrip * ((g.ny + rows - 1) / rows);
        const double cost = (double)((items + slots - 1) / slots) * (rows + 3.0);
        if (cost < best_cost - 1e-9) { best_cost = cost; best = rows; }
    }
    return best;
}

template <int STAGE>
inline cudaError_t launch_stage_warp2d(const Grid &g, const double *in, const double *old, double *out, double r,
                                       const StepScalars *dev_dt, double dx, StepScalars *red, int rows,
                                       cudaStream_t stream)
{
    Warp2dArgs a;
    a.g = g; a.Uin = in; a.Uold = old; a.Uout = out; a.dt_over_dx = r; a.dev_dt = dev_dt; a.dx = dx; a.red = red;
    a.rows = rows < 1 ? 1 : (rows > g.ny ? g.ny : rows);
    a.nstrip = (g.nx + W2_OWN - 1) / W2_OWN;
    a.nchunk = (g.ny + a.rows - 1) / a.rows;
    const unsigned blocks = (unsigned)(((long long)a.nstrip * a.nchunk + W2_WARPS - 1) / W2_WARPS);
    if (g.ry != 1.0) stage_warp2d_kernel<STAGE, true><<<blocks, 32 * W2_WARPS, 0, stream>>>(a);
    else             stage_warp2d_kernel<STAGE, false><<<blocks, 32 * W2_WARPS, 0, stream>>>(a);
    return cudaGetLastError();
}

}  // namespace hyd
