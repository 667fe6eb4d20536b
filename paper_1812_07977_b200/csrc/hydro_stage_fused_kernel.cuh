// hydro_stage_fused_kernel.cuh -- body of the fused stage kernel (see hydro_stage_fused.cuh).
#pragma once
#include <cstdlib>

namespace hyd {

struct FusedArgs {
    Grid g;
    const double *Uin;      // stencil input (stage 1: U0, stage 2: U1), ghost-filled
    const double *Uold;     // stage 2: U0 (read at the thread's own cell only); may alias Uout
    double *Uout;
    double dt_over_dx;      // used when dev_dt == nullptr
    const StepScalars *dev_dt;
    double dx;
    StepScalars *red;       // stage 2: max-signal-speed accumulator + sticky flag (or nullptr)
    int lz;                 // planes per z-chunk
};

template <int STAGE, int TY, int MINB>
__global__ void __launch_bounds__(FTX * TY, MINB)
stage_fused_kernel(const FusedArgs a)
{
    using S = FusedSmem<TY>;
    constexpr int TX = FTX, WP = S::WP, XP = S::XP;
    extern __shared__ __align__(16) double sm[];
    double *Wsm = sm + S::OFF_W, *Oxs = sm + S::OFF_OX, *Oys = sm + S::OFF_OY;
    double *Fxs = sm + S::OFF_FX, *Fys = sm + S::OFF_FY;
    double *Ixe = sm + S::OFF_IXE, *Iye = sm + S::OFF_IYE;

    const Grid &g = a.g;
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * TX + tx;
    const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;     // tile origin, active coordinates
    const int k0 = blockIdx.z * a.lz;
    const int k1 = min(k0 + a.lz, g.nz);                      // chunk = active planes [k0, k1)
    const int Imax = g.nx + 3, Jmax = g.ny + 3;
    const double gamma = g.gamma, gm1 = g.gm1, igm1 = g.igm1, theta = g.theta;
    const long long sv = g.sv, sy = g.sy;

    // own column: padded (I, J); threads past the active range still compute (they own the
    // domain's high-edge faces) but never write global memory
    const int I = min(i0 + tx + NG, Imax), J = min(j0 + ty + NG, Jmax);
    const bool active = (i0 + tx < g.nx) && (j0 + ty < g.ny);
    const long long col = (long long)I + (long long)g.px * J;
    const int wc = (ty + 2) * WP + tx + 2;                    // own cell in the primitive tile

    // halo cell of this thread (first 4*TY + 4*TX threads), tile coordinates (hc, hr)
    constexpr int NHX = 4 * TY, NH = 4 * TY + 4 * TX;
    int hc = 0, hr = 0;
    if (t < NHX) { const int q = t & 3; hr = (t >> 2) + 2; hc = q < 2 ? q : TX + q; }
    else if (t < NH) { const int u = t - NHX, q = u / TX; hc = (u % TX) + 2; hr = q < 2 ? q : TY + q; }
    const bool has_halo = t < NH;
    const long long hcol = (long long)min(i0 + hc, Imax) + (long long)g.px * min(j0 + hr, Jmax);
    const int hw = hr * WP + hc;

    const double r = a.dev_dt ? a.dev_dt->dt / a.dx : a.dt_over_dx;

    double Wa[5], Wb[5];          // W(kk-2), W(kk-1)
    double Oz[5];                 // outer z-face value of cell kk-2
    double Fzm[5];                // flux through face (kk-2)-1/2
    double smax = 0.0;
    int bad = 0;
#pragma unroll
    for (int v = 0; v < 5; ++v) { Wa[v] = Wb[v] = Oz[v] = Fzm[v] = 0.0; }

    double Un[5], Uh[5];
    load5(a.Uin, sv, col + sy * (long long)(k0 - 2 + NG), Un);
#pragma unroll
    for (int v = 0; v < 5; ++v) Uh[v] = 1.0;

#pragma unroll 1
    for (int kk = k0 - 2; kk < k1 + 2; ++kk) {
        const bool do_slope = kk >= k0, do_flux = kk >= k0 + 1, do_cell = kk >= k0 + 2;
        // ---------------- phase 1: primitives of the new plane; z pipeline -------------------
        double Wn[5];
        HYD_PRIM5(Un, gm1, Wn);
        if (kk + 1 < k1 + 2) load5(a.Uin, sv, col + sy * (long long)(kk + 1 + NG), Un);
        double dFz[5];
        if (do_slope) {
            double Iz[5], Ozn[5];
            HYD_LIMITED_FACES(theta, Wa, Wb, Wn, Iz, Ozn);        // cell kk-1
            if (do_flux) {
                double Fzp[5];
                face_flux<2>(Oz, Iz, gamma, igm1, Fzp);       // face (kk-2)+1/2
#pragma unroll
                for (int v = 0; v < 5; ++v) { dFz[v] = Fzp[v] - Fzm[v]; Fzm[v] = Fzp[v]; }
            }
#pragma unroll
            for (int v = 0; v < 5; ++v) Oz[v] = Ozn[v];
        }
        double Wc[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) { Wc[v] = Wa[v]; Wa[v] = Wb[v]; Wb[v] = Wn[v]; }
        if (!do_cell) {
            // the first cell plane of the chunk is two iterations ahead: fetch its halo
            if (kk + 1 >= k0 + 2 && has_halo) load5(a.Uin, sv, hcol + sy * (long long)(kk - 1 + NG), Uh);
            continue;
        }
        const int k = kk - 2;                                 // the plane completed this iteration
        const long long cg = col + sy * (long long)(k + NG);
#pragma unroll
        for (int v = 0; v < 5; ++v) Wsm[v * S::WSZ + wc] = Wc[v];
        if (has_halo) {
            double Wh[5];
            HYD_PRIM5(Uh, gm1, Wh);
#pragma unroll
            for (int v = 0; v < 5; ++v) Wsm[v * S::WSZ + hw] = Wh[v];
            if (k + 1 < k1) load5(a.Uin, sv, hcol + sy * (long long)(k + 1 + NG), Uh);
        }
        __syncthreads();
        // ---------------- phase 2: x and y slopes, face values -------------------------------
        double Ix[5], Iy[5];
        {
            double Wm[5], Wp[5], Ox[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wm[v] = Wsm[v * S::WSZ + wc - 1]; Wp[v] = Wsm[v * S::WSZ + wc + 1]; }
            HYD_LIMITED_FACES(theta, Wm, Wc, Wp, Ix, Ox);
#pragma unroll
            for (int v = 0; v < 5; ++v) Oxs[v * S::XSZ + ty * XP + tx + 1] = Ox[v];
        }
        {
            double Wm[5], Wp[5], Oy[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wm[v] = Wsm[v * S::WSZ + wc - WP]; Wp[v] = Wsm[v * S::WSZ + wc + WP]; }
            HYD_LIMITED_FACES(theta, Wm, Wc, Wp, Iy, Oy);
#pragma unroll
            for (int v = 0; v < 5; ++v) Oys[v * S::YSZ + (ty + 1) * TX + tx] = Oy[v];
        }
        // halo-cell slopes: x: cells (-1, j) -> outer, (TX, j) -> inner; y: rows -1 -> outer, TY -> inner
        if (t < 2 * TY + 2 * TX) {
            int c, st, dst;
            bool want_outer;
            if (t < 2 * TY) {
                const int j = t >> 1, hi = t & 1;
                c = (j + 2) * WP + (hi ? TX + 2 : 1); st = 1; want_outer = !hi;
                dst = hi ? S::OFF_IXE + j : S::OFF_OX + j * XP;
            } else {
                const int u = t - 2 * TY, hi = u / TX, i = u % TX;
                c = (hi ? TY + 2 : 1) * WP + i + 2; st = WP; want_outer = !hi;
                dst = hi ? S::OFF_IYE + i : S::OFF_OY + i;
            }
            const int dstride = t < 2 * TY ? ((t & 1) ? TY : S::XSZ) : ((t - 2 * TY) / TX ? TX : S::YSZ);
            double Wm[5], W0[5], Wp[5], In[5], Ou[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                Wm[v] = Wsm[v * S::WSZ + c - st]; W0[v] = Wsm[v * S::WSZ + c]; Wp[v] = Wsm[v * S::WSZ + c + st];
            }
            HYD_LIMITED_FACES(theta, Wm, W0, Wp, In, Ou);
#pragma unroll
            for (int v = 0; v < 5; ++v) sm[dst + v * dstride] = want_outer ? Ou[v] : In[v];
        }
        __syncthreads();
        // ---------------- phase 3: x and y fluxes through the low faces ----------------------
        double Fxl[5], Fyl[5];
        {
            double L[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) L[v] = Oxs[v * S::XSZ + ty * XP + tx];
            face_flux<0>(L, Ix, gamma, igm1, Fxl);
#pragma unroll
            for (int v = 0; v < 5; ++v) Fxs[v * S::XSZ + ty * XP + tx] = Fxl[v];
        }
        {
            double L[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) L[v] = Oys[v * S::YSZ + ty * TX + tx];
            face_flux<1>(L, Iy, gamma, igm1, Fyl);
#pragma unroll
            for (int v = 0; v < 5; ++v) Fys[v * S::YSZ + ty * TX + tx] = Fyl[v];
        }
        // the tile's high-edge faces: warp 0 lanes < TY: x face TX-1/2+1 of row `lane`;
        // warp 1: y face of column `lane`
        if (ty == 0 && tx < TY) {
            double L[5], R[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { L[v] = Oxs[v * S::XSZ + tx * XP + TX]; R[v] = Ixe[v * TY + tx]; }
            face_flux<0>(L, R, gamma, igm1, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) Fxs[v * S::XSZ + tx * XP + TX] = F[v];
        } else if (ty == 1) {
            double L[5], R[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { L[v] = Oys[v * S::YSZ + TY * TX + tx]; R[v] = Iye[v * TX + tx]; }
            face_flux<1>(L, R, gamma, igm1, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) Fys[v * S::YSZ + TY * TX + tx] = F[v];
        }
        __syncthreads();
        // ---------------- phase 4: divergence, RK combine, store, CFL ------------------------
        double un[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double dFx = Fxs[v * S::XSZ + ty * XP + tx + 1] - Fxl[v];
            const double dFy = Fys[v * S::YSZ + (ty + 1) * TX + tx] - Fyl[v];
            const double D = HYD_SUM3(dFx, dFy, dFz[v]);
            const double dU = -(r * D);
            if (STAGE == 1) {
                un[v] = __ldg(a.Uin + v * sv + cg) + dU;
            } else {
                const double sum = a.Uold[v * sv + cg] + __ldg(a.Uin + v * sv + cg);
                un[v] = 0.5 * (sum + dU);
            }
        }
        if (active) {
#pragma unroll
            for (int v = 0; v < 5; ++v) a.Uout[v * sv + cg] = un[v];
            if (STAGE == 2 && a.red) {
                const double s = cell_signal_speed(un[0], un[1], un[2], un[3], un[4], gamma, gm1, bad);
                smax = s > smax ? s : smax;
            }
        }
    }
    if (STAGE == 2 && a.red) block_max_to_global(smax, bad, &a.red->smax_bits, &a.red->flag);
}

// ------------------------------------------------------------------------------------------
// host side: launch geometry
// ------------------------------------------------------------------------------------------
struct FusedPlan {
    int ready = 0;
    int ty = 16;             // tile height (8 or 16)
    int lz = 32;             // planes per z-chunk
    dim3 grid;
};

template <int STAGE, int TY, int MINB>
inline cudaError_t fused_set_attr()
{
    return cudaFuncSetAttribute(stage_fused_kernel<STAGE, TY, MINB>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)FusedSmem<TY>::BYTES);
}

inline void fused_geometry(FusedPlan &p, const Grid &g, int ty, int lz)
{
    p.ty = ty;
    p.lz = lz < 1 ? 1 : (lz > g.nz ? g.nz : lz);
    p.grid = dim3((g.nx + FTX - 1) / FTX, (g.ny + ty - 1) / ty, (g.nz + p.lz - 1) / p.lz);
}

inline cudaError_t plan_stage_fused(FusedPlan &p, const Grid &g, const double *, const double *)
{
    cudaError_t e;
    if ((e = fused_set_attr<1, 16, 1>()) != cudaSuccess) return e;
    if ((e = fused_set_attr<2, 16, 1>()) != cudaSuccess) return e;
    if ((e = fused_set_attr<1, 8, 2>()) != cudaSuccess) return e;
    if ((e = fused_set_attr<2, 8, 2>()) != cudaSuccess) return e;
    int nsm = 148;
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess)
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    // tuning knobs (measurement only): HYDRO_FUSED_TY = 8 | 16, HYDRO_FUSED_LZ = planes per chunk
    const char *ety = getenv("HYDRO_FUSED_TY"), *elz = getenv("HYDRO_FUSED_LZ");
    const int ty = (ety && atoi(ety) == 16) ? 16 : 8;
    const int per_sm = ty == 16 ? 1 : 2;
    // choose lz so that the block count fills whole waves of nsm * per_sm blocks as evenly as
    // possible while keeping the two warm-up planes per chunk a small overhead
    const long long tiles = (long long)((g.nx + FTX - 1) / FTX) * ((g.ny + ty - 1) / ty);
    int best = g.nz;
    double best_cost = 1e300;
    for (int lz = 4; lz <= g.nz || lz == 4; ++lz) {
        const int l = lz > g.nz ? g.nz : lz;
        const long long chunks = (g.nz + l - 1) / l;
        const long long blocks = tiles * chunks;
        const long long waves = (blocks + (long long)nsm * per_sm - 1) / ((long long)nsm * per_sm);
        // time ~ waves * (planes per block incl. warm-up), in plane units
        const double cost = (double)waves * (l + 4);
        if (cost < best_cost - 1e-9) { best_cost = cost; best = l; }
        if (lz > g.nz) break;
    }
    if (elz && atoi(elz) > 0) best = atoi(elz);
    fused_geometry(p, g, ty, best);
    p.ready = 1;
    return cudaSuccess;
}

template <int STAGE>
inline cudaError_t launch_stage_fused(const FusedPlan &p, const Grid &g, const double *in,
                                      const double *old, double *out, double r,
                                      const StepScalars *dev_dt, double dx, StepScalars *red,
                                      cudaStream_t stream)
{
    FusedArgs a;
    a.g = g; a.Uin = in; a.Uold = old; a.Uout = out; a.dt_over_dx = r; a.dev_dt = dev_dt; a.dx = dx;
    a.red = red; a.lz = p.lz;
    if (p.ty == 16)
        stage_fused_kernel<STAGE, 16, 1><<<p.grid, dim3(FTX, 16), FusedSmem<16>::BYTES, stream>>>(a);
    else
        stage_fused_kernel<STAGE, 8, 2><<<p.grid, dim3(FTX, 8), FusedSmem<8>::BYTES, stream>>>(a);
    return cudaGetLastError();
}

}  // namespace hyd
