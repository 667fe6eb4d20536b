// hydro_stage_fused_kernel.cuh -- body of the fused stage kernel (see hydro_stage_fused.cuh).
#pragma once
#include <cstdlib>

namespace hyd {

struct FusedArgs {
    Grid g;
    const double *Uold;     // stage 2: U0 (read at the thread's own cell only); may alias Uout
    double *Uout;
    double dt_over_dx;      // used when dev_dt == nullptr
    const StepScalars *dev_dt;
    double dx;
    StepScalars *red;       // stage 2: max-signal-speed accumulator + sticky flag (or nullptr)
    int lz;                 // planes per z-chunk
};

// `umap` describes the stencil input (stage 1: U0, stage 2: U1; ghost-filled) to the TMA unit.
template <int STAGE, int TY, int MINB>
__global__ void __launch_bounds__(FTX * TY, MINB)
stage_fused_kernel(const __grid_constant__ CUtensorMap umap, const FusedArgs a)
{
    using S = FusedSmem<TY>;
    constexpr int TX = FTX, WP = S::WP, XP = S::XP;
    extern __shared__ __align__(128) double sm[];
    double *Wsm = sm + S::OFF_W, *Oxs = sm + S::OFF_OX, *Oys = sm + S::OFF_OY;
    double *Fxs = sm + S::OFF_FX, *Fys = sm + S::OFF_FY;
    double *Ixe = sm + S::OFF_IXE, *Iye = sm + S::OFF_IYE;
    uint64_t *bar = reinterpret_cast<uint64_t *>(sm + S::OFF_BAR);

    const Grid &g = a.g;
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * TX + tx;
    const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;     // tile origin, active coordinates
    const int k0 = blockIdx.z * a.lz;
    const int k1 = min(k0 + a.lz, g.nz);                      // chunk = active planes [k0, k1)
    const int nplanes = k1 - k0 + 4;                          // planes k0-2 .. k1+1 stream through
    const double gamma = g.gamma, gm1 = g.gm1, igm1 = g.igm1, theta = g.theta;
    const long long sv = g.sv;

    // own column; threads past the active range still compute (they own the domain's high-edge
    // faces) but never touch global memory
    const bool active = (i0 + tx < g.nx) && (j0 + ty < g.ny);
    const long long col = (long long)(i0 + tx + NG) + (long long)g.px * (j0 + ty + NG);
    const int wc = (ty + 2) * WP + tx + 2;                    // own cell in a (tile + halo) plane

    // halo cell of this thread (first 4*TY + 4*TX threads), plane coordinates (hc, hr)
    constexpr int NHX = 4 * TY, NH = 4 * TY + 4 * TX;
    int hc = 0, hr = 0;
    if (t < NHX) { const int q = t & 3; hr = (t >> 2) + 2; hc = q < 2 ? q : TX + q; }
    else if (t < NH) { const int u = t - NHX, q = u / TX; hc = (u % TX) + 2; hr = q < 2 ? q : TY + q; }
    const bool has_halo = t < NH;
    const int hw = hr * WP + hc;

    // ---- TMA ring: plane index p (0 = active plane k0-2) lives in stage p % FNS ----------------
    if (t == 0) {
#pragma unroll
        for (int s = 0; s < FNS; ++s) tma::mbar_init(&bar[s], 1);
        tma::fence_barrier_init();
    }
    __syncthreads();
    if (t == 0) {
        const int np = nplanes < FNS ? nplanes : FNS;
        for (int p = 0; p < np; ++p) {
            tma::mbar_arrive_expect_tx(&bar[p], S::STAGE_BYTES);
            tma::load_4d(sm + S::OFF_RING + p * S::STAGE, &umap, i0, j0, k0 + p, 0, &bar[p]);
        }
    }

    const double r = a.dev_dt ? a.dev_dt->dt / a.dx : a.dt_over_dx;

    double Wa[5], Wb[5];          // W(kk-2), W(kk-1)
    double Oz[5];                 // outer z-face value of cell kk-2
    double Fzm[5];                // flux through face (kk-2)-1/2
    double smax = 0.0;
    int bad = 0;
#pragma unroll
    for (int v = 0; v < 5; ++v) { Wa[v] = Wb[v] = Oz[v] = Fzm[v] = 0.0; }

#pragma unroll 1
    for (int p = 0; p < nplanes; ++p) {
        const int kk = k0 - 2 + p;
        const bool do_slope = p >= 2, do_flux = p >= 3, do_cell = p >= 4;
        const double *Ucur = sm + S::OFF_RING + (p % FNS) * S::STAGE;          // raw plane kk
        const double *Uk = sm + S::OFF_RING + ((p + 2) % FNS) * S::STAGE;      // raw plane kk-2
        tma::mbar_wait(&bar[p % FNS], (p / FNS) & 1);
        // ---------------- phase 1: primitives of the new plane; z pipeline -------------------
        double Wn[5];
        {
            double Un[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) Un[v] = Ucur[v * S::WSZ + wc];
            HYD_PRIM5(Un, gm1, Wn);
        }
        double dFz[5];
        if (do_slope) {
            double Iz[5], Ozn[5];
            HYD_LIMITED_FACES(theta, Wa, Wb, Wn, Iz, Ozn);    // cell kk-1
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
        if (do_cell) {
#pragma unroll
            for (int v = 0; v < 5; ++v) Wsm[v * S::WSZ + wc] = Wc[v];
            if (has_halo) {
                double Uh[5], Wh[5];
#pragma unroll
                for (int v = 0; v < 5; ++v) Uh[v] = Uk[v * S::WSZ + hw];
                HYD_PRIM5(Uh, gm1, Wh);
#pragma unroll
                for (int v = 0; v < 5; ++v) Wsm[v * S::WSZ + hw] = Wh[v];
            }
        }
        __syncthreads();
        // every thread is past its reads of plane p-3 (stage (p+1) % FNS): refill it with p+1
        if (t == 0 && p + 1 >= FNS && p + 1 < nplanes) {
            tma::fence_proxy_async();
            tma::mbar_arrive_expect_tx(&bar[(p + 1) % FNS], S::STAGE_BYTES);
            tma::load_4d(sm + S::OFF_RING + ((p + 1) % FNS) * S::STAGE, &umap, i0, j0, k0 + p + 1, 0,
                         &bar[(p + 1) % FNS]);
        }
        if (!do_cell) continue;
        const int k = kk - 2;                                 // the plane completed this iteration
        const long long cg = col + g.sy * (long long)(k + NG);
        if (STAGE == 2 && active) {
#pragma unroll
            for (int v = 0; v < 5; ++v)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Uold + v * sv + cg));
        }
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
            int c, st, dst, dstride;
            bool want_outer;
            if (t < 2 * TY) {
                const int j = t >> 1, hi = t & 1;
                c = (j + 2) * WP + (hi ? TX + 2 : 1); st = 1; want_outer = !hi;
                dst = hi ? S::OFF_IXE + j : S::OFF_OX + j * XP;
                dstride = hi ? TY : S::XSZ;
            } else {
                const int u = t - 2 * TY, hi = u / TX, i = u % TX;
                c = (hi ? TY + 2 : 1) * WP + i + 2; st = WP; want_outer = !hi;
                dst = hi ? S::OFF_IYE + i : S::OFF_OY + i;
                dstride = hi ? TX : S::YSZ;
            }
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
        // the tile's high-edge faces: warp 0 lanes < TY: x face of row `lane`; warp 1: y face of
        // column `lane` (each flux is written over the outer value it consumed)
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
        double Uo[5];
        if (STAGE == 2) {                                     // in flight across the barrier
#pragma unroll
            for (int v = 0; v < 5; ++v) Uo[v] = active ? a.Uold[v * sv + cg] : 0.0;
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
            const double u1 = Uk[v * S::WSZ + wc];
            if (STAGE == 1) {
                un[v] = u1 + dU;
            } else {
                const double sum = Uo[v] + u1;
                un[v] = 0.5 * (sum + dU);
            }
        }
        if (active) {
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
    if (STAGE == 2 && a.red) {
        if (!(smax <= 1.79769313486231570e308)) { bad = 1; smax = 0.0; }   // inf or NaN pattern won
        block_max_to_global(smax, bad, &a.red->smax_bits, &a.red->flag);
    }
}

}  // namespace hyd

#include "hydro_stage_fused_plan.cuh"
