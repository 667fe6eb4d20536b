// hydro_stage_fused2d.cuh -- the fused RK-stage kernel of 2D runs (hydro_create_nd, ndim = 2;
// PAPER.md:134, 138; R21-R23).
//
// Same building blocks, shared-memory carve-up and hand-off scheme as the 3D kernel
// (hydro_stage_fused_kernel.cuh, 32 x 16 tiles, "PIPE" flow), with the march turned sideways: there
// is no z axis, so a block owns a column of 32 cells in x and walks DOWN y, one 32 x 16 tile per
// iteration.  The degenerate axis issues no loads, slopes or fluxes.  Every tile (plus its 2-cell
// halo) arrives through the same TMA ring; the primitives of tile c+1 (own cells and halo) are formed
// while tile c is being updated, so one flux barrier carries both hand-offs:
//   per tile c:  y-slopes, halo slopes  arrive_O  [x-slopes, primitives of the own cell of tile c+1]
//                wait_O  tile(c+1), x/y fluxes, edge fluxes  arrive_F  wait_F  update
// No register pipeline (nothing is carried between tiles but the own primitives of the next one),
// boundary rules in the kernel as in 3D (outflow / reflecting x, y from the source cell; periodic
// axes from memory ghosts that the update keeps current).
#pragma once
#include "hydro_stage_fused.cuh"

namespace hyd {

template <int STAGE, bool ANISO, bool WRAP>
__global__ void __launch_bounds__(FTX * 16, 1)
stage_fused2d_kernel(const __grid_constant__ CUtensorMap umap, const FusedArgs a)
{
    constexpr int TY = 16;
    using S = FusedSmem<TY>;
    constexpr int TX = FTX, WP = S::WP, XP = S::XP;
    extern __shared__ __align__(128) double sm[];
    double *Oxs = sm + S::OFF_OX, *Oys = sm + S::OFF_OY;
    double *Fxs = sm + S::OFF_FX, *Fys = sm + S::OFF_FY;
    double *Ixe = sm + S::OFF_IXE, *Iye = sm + S::OFF_IYE;
    uint64_t *bar = reinterpret_cast<uint64_t *>(sm + S::OFF_BAR);     // TMA: tile p -> bar[p % FNS]
    uint64_t *barO = bar + FNS + 1, *barF = bar + FNS + 2;

    const Grid &g = a.g;
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * TX + tx;
    const int i0 = blockIdx.x * TX;
    const int ntile = (g.ny + TY - 1) / TY;                   // tile rows of the grid
    const int t0 = blockIdx.y * a.lz;                         // this block's chunk: tile rows [t0, t0 + nc)
    const int nc = min(t0 + a.lz, ntile) - t0;
    const double gamma = g.gamma, gm1 = g.gm1, igm1 = g.igm1, theta = g.theta;
    const long long sv = g.sv;
    const int wc = (ty + 2) * WP + tx + 2;                    // own cell in a (tile + halo) plane
    constexpr int NHX = 4 * TY, NH = 4 * TY + 4 * TX;

    // conserved state of the own cell of the tile with y origin j0 (boundary rule applied for the
    // threads that stand in for ghost cells of the high faces)
    auto load_own = [&](const double *Ust, int j0, double Un[5]) {
        int ws = wc;
        bool fx = false, fy = false;
        const bool actv = (i0 + tx < g.nx) && (j0 + ty < g.ny);
        if (!actv && (a.inbc & 3)) {
            const int is = (a.inbc & 1) ? bc_source(i0 + tx, g.nx, g.bc[0], g.bc[1], i0 - NG, i0 + TX + NG - 1, fx) : i0 + tx;
            const int js = (a.inbc & 2) ? bc_source(j0 + ty, g.ny, g.bc[2], g.bc[3], j0 - NG, j0 + TY + NG - 1, fy) : j0 + ty;
            ws = (js - j0 + NG) * WP + (is - i0 + NG);
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) Un[v] = Ust[v * S::WSZ + ws];
        if (!actv) { Un[1] = flip_sign(Un[1], fx); Un[2] = flip_sign(Un[2], fy); }
    };

    if (t == 0) {
#pragma unroll
        for (int s = 0; s < FNS; ++s) tma::mbar_init(&bar[s], 1);
        tma::mbar_init(barO, TY); tma::mbar_init(barF, TY);
        tma::fence_barrier_init();
    }
    __syncthreads();
    auto request_tile = [&](int p) {                          // thread 0 only
        tma::mbar_arrive_expect_tx(&bar[p % FNS], S::STAGE_BYTES);
        tma::load_4d(sm + S::OFF_RING + (p % FNS) * S::STAGE, &umap, i0, (t0 + p) * TY, 0, 0, &bar[p % FNS]);
    };
    if (t == 0)
        for (int p = 0; p < FNS && p < nc; ++p) request_tile(p);

    const double r = a.dev_dt ? a.dev_dt->dt / a.dx : a.dt_over_dx;

    // primitive tile: own cell from registers, halo cells from the raw tile (boundary rule applied)
    auto write_tile = [&](double *Wsm, const double Wown[5], const double *Uraw, int role, int j0) {
#pragma unroll
        for (int v = 0; v < 5; ++v) Wsm[v * S::WSZ + wc] = Wown[v];
        const int th = (role - 3) * TX + tx;
        if (th >= 0 && th < NH) {
            int hc, hr;
            if (th < NHX) { const int q = th & 3; hr = (th >> 2) + 2; hc = q < 2 ? q : TX + q; }
            else { const int u = th - NHX, q = u / TX; hc = (u % TX) + 2; hr = q < 2 ? q : TY + q; }
            const int hw = hr * WP + hc;
            int hs = hw;
            bool fx = false, fy = false;
            const bool edge_tile = ((a.inbc & 1) && (i0 == 0 || i0 + TX + NG > g.nx)) ||
                                   ((a.inbc & 2) && (j0 == 0 || j0 + TY + NG > g.ny));
            if (edge_tile) {
                const int is = (a.inbc & 1) ? bc_source(i0 + hc - NG, g.nx, g.bc[0], g.bc[1], i0 - NG, i0 + TX + NG - 1, fx) : i0 + hc - NG;
                const int js = (a.inbc & 2) ? bc_source(j0 + hr - NG, g.ny, g.bc[2], g.bc[3], j0 - NG, j0 + TY + NG - 1, fy) : j0 + hr - NG;
                hs = (js - j0 + NG) * WP + (is - i0 + NG);
            }
            double Uh[5], Wh[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) Uh[v] = Uraw[v * S::WSZ + hs];
            if (edge_tile) { Uh[1] = flip_sign(Uh[1], fx); Uh[2] = flip_sign(Uh[2], fy); }
            HYD_PRIM5(Uh, gm1, Wh);
#pragma unroll
            for (int v = 0; v < 5; ++v) Wsm[v * S::WSZ + hw] = Wh[v];
        }
    };

    // ---- prologue: primitives of tile 0 ---------------------------------------------------------
    double Wa[5], Wn[5];
    double smax = 0.0;
    int bad = 0;
#pragma unroll
    for (int v = 0; v < 5; ++v) Wa[v] = Wn[v] = 0.0;
    if (nc > 0) {
        tma::mbar_wait(&bar[0], 0);
        double Un[5];
        load_own(sm + S::OFF_RING, t0 * TY, Un);
        HYD_PRIM5(Un, gm1, Wa);
        write_tile(sm + S::OFF_W, Wa, sm + S::OFF_RING, ty, t0 * TY);
    }
    __syncthreads();

#pragma unroll 1
    for (int c = 0; c < nc; ++c) {
        const uint32_t par = c & 1;
        const int role = (ty + c) & (TY - 1);
        const int j0 = (t0 + c) * TY;
        const bool active = (i0 + tx < g.nx) && (j0 + ty < g.ny);
        const double *Uk = sm + S::OFF_RING + (c % FNS) * S::STAGE;            // raw tile c
        const long long cg = (long long)(i0 + tx + NG) + (long long)g.px * (j0 + ty + NG);
        double *Wsm = sm + S::OFF_W + (c & 1) * S::STAGE;
        // ---- y-slopes of the own cell, halo-cell slopes ------------------------------------------
        double Ix[5], Iy[5];
        {
            double Wm[5], Wp[5], Oy[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wm[v] = Wsm[v * S::WSZ + wc - WP]; Wp[v] = Wsm[v * S::WSZ + wc + WP]; }
            HYD_LIMITED_FACES(theta, Wm, Wa, Wp, Iy, Oy);
#pragma unroll
            for (int v = 0; v < 5; ++v) Oys[v * S::YSZ + (ty + 1) * TX + tx] = Oy[v];
        }
        if (role == 2 || role == 3 || (role == 6 && tx < 2 * TY) || (role == 7 && tx < TY)) {
            int cc, st, dst, dstride;
            bool want_outer;
            if (role == 6) {
                const int j = tx >> 1, hi = tx & 1;
                cc = (j + 2) * WP + (hi ? TX + 2 : 1); st = 1; want_outer = !hi;
                dst = hi ? S::OFF_IXE + j : S::OFF_OX + j * XP;
                dstride = hi ? TY : S::XSZ;
            } else if (role == 7) {
                cc = (tx + 2) * WP + TX + 1; st = 1; want_outer = true;
                dst = S::OFF_OXE + (c & 1) * NVAR * TY + tx; dstride = TY;
            } else {
                const int hi = role - 2, i = tx;
                cc = (hi ? TY + 2 : 1) * WP + i + 2; st = WP; want_outer = !hi;
                dst = hi ? S::OFF_IYE + i : S::OFF_OY + i;
                dstride = hi ? TX : S::YSZ;
            }
            double Wm[5], W0[5], Wp[5], In[5], Ou[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                Wm[v] = Wsm[v * S::WSZ + cc - st]; W0[v] = Wsm[v * S::WSZ + cc]; Wp[v] = Wsm[v * S::WSZ + cc + st];
            }
            HYD_LIMITED_FACES(theta, Wm, W0, Wp, In, Ou);
#pragma unroll
            for (int v = 0; v < 5; ++v) sm[dst + v * dstride] = want_outer ? Ou[v] : In[v];
        }
        __syncwarp();
        if (tx == 0) tma::mbar_arrive(barO);
        // ---- filler: own x-slopes (stay inside the warp), own primitives of the next tile ----------
        {
            double Wm[5], Wp[5], Ox[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wm[v] = Wsm[v * S::WSZ + wc - 1]; Wp[v] = Wsm[v * S::WSZ + wc + 1]; }
            HYD_LIMITED_FACES(theta, Wm, Wa, Wp, Ix, Ox);
            if (tx != TX - 1) {
#pragma unroll
                for (int v = 0; v < 5; ++v) Oxs[v * S::XSZ + ty * XP + tx + 1] = Ox[v];
            }
        }
        if (c + 1 < nc) {
            const int p = c + 1;
            tma::mbar_wait(&bar[p % FNS], (p / FNS) & 1);
            double Un[5];
            load_own(sm + S::OFF_RING + (p % FNS) * S::STAGE, (t0 + p) * TY, Un);
            HYD_PRIM5(Un, gm1, Wn);
        }
        tma::mbar_wait_sync(barO, par);
        __syncwarp();
        // every warp is past the update of tile c-1: its raw tile is dead, refill that stage
        if (t == 0 && c >= 1 && c + 3 < nc) { tma::fence_proxy_async(); request_tile(c + 3); }
        // ---- primitive tile of tile c+1, x and y fluxes through the low faces ----------------------
        double Fxl[5], Fyl[5];
        if (c + 1 < nc)
            write_tile(sm + S::OFF_W + ((c + 1) & 1) * S::STAGE, Wn,
                       sm + S::OFF_RING + ((c + 1) % FNS) * S::STAGE, (ty + c + 1) & (TY - 1), (t0 + c + 1) * TY);
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
        if (role == 0 && tx < TY) {
            double L[5], R[5], F[5];
            const double *Le = sm + S::OFF_OXE + (c & 1) * NVAR * TY + tx;
#pragma unroll
            for (int v = 0; v < 5; ++v) { L[v] = Le[v * TY]; R[v] = Ixe[v * TY + tx]; }
            face_flux<0>(L, R, gamma, igm1, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) Fxs[v * S::XSZ + tx * XP + TX] = F[v];
        } else if (role == 1) {
            double L[5], R[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { L[v] = Oys[v * S::YSZ + TY * TX + tx]; R[v] = Iye[v * TX + tx]; }
            face_flux<1>(L, R, gamma, igm1, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) Fys[v * S::YSZ + TY * TX + tx] = F[v];
        }
        __syncwarp();
        if (tx == 0) tma::mbar_arrive(barF);
        double Uo[5];
        if (STAGE == 2) {
#pragma unroll
            for (int v = 0; v < 5; ++v) Uo[v] = active ? a.Uold[v * sv + cg] : 0.0;
        }
        tma::mbar_wait_sync(barF, par);
        // ---- divergence (O5, two dimensions: D = dFx + (dx/dy) dFy), RK combine, store, CFL --------
        double un[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double dFx = Fxs[v * S::XSZ + ty * XP + tx + 1] - Fxl[v];
            double dFy = Fys[v * S::YSZ + (ty + 1) * TX + tx] - Fyl[v];
            if (ANISO) dFy = g.ry * dFy;
            const double D = dFx + dFy;
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
            if (WRAP) {         // periodic x / y: the producer also writes the ghost images of its cell
                const int i = i0 + tx, j = j0 + ty;
                if ((a.wrap & 1) && i < NG) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) a.Uout[v * sv + cg + g.nx] = un[v];
                }
                if ((a.wrap & 1) && i >= g.nx - NG) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) a.Uout[v * sv + cg - g.nx] = un[v];
                }
                if ((a.wrap & 2) && j < NG) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) a.Uout[v * sv + cg + (long long)g.px * g.ny] = un[v];
                }
                if ((a.wrap & 2) && j >= g.ny - NG) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) a.Uout[v * sv + cg - (long long)g.px * g.ny] = un[v];
                }
            }
            if (STAGE == 2 && a.red) {
#ifdef HYDRO_VERIFY
                const double s = cell_signal_speed(un[0], un[1], un[2], un[3], un[4], gamma, gm1, bad);
                smax = s > smax ? s : smax;
#else
                smax = fast::max_nonneg(smax, fast::signal_speed(un, gamma, gm1, bad));
#endif
            }
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) Wa[v] = Wn[v];
    }
    if (STAGE == 2 && a.red) {
        if (!(smax <= 1.79769313486231570e308)) { bad = 1; smax = 0.0; }
        block_max_to_global(smax, bad, &a.red->smax_bits, &a.red->flag);
    }
}

// ---- host side ------------------------------------------------------------------------------------

// tile rows per block: whole waves of one block per SM; a chunk of l tiles costs about (l + 1) tile times
inline int fused2d_choose_lz(const Grid &g, int nsm)
{
    const long long tx = (g.nx + FTX - 1) / FTX;
    const int ntile = (g.ny + 15) / 16;
    int best = ntile;
    double best_cost = 1e300;
    for (int l = ntile; l >= 1; --l) {
        const long long blocks = tx * ((ntile + l - 1) / l);
        const long long waves = (blocks + nsm - 1) / nsm;
        const double cost = (double)waves * (l + 1);
        if (cost < best_cost - 1e-9) { best_cost = cost; best = l; }
    }
    return best;
}

inline cudaError_t plan_stage_fused2d(FusedPlan &p, const Grid &g, const double *A, const double *B, int lz_req = 0)
{
    cudaError_t e;
    const void *fns[8] = { (const void *)stage_fused2d_kernel<1, false, false>, (const void *)stage_fused2d_kernel<1, true, false>,
                           (const void *)stage_fused2d_kernel<2, false, false>, (const void *)stage_fused2d_kernel<2, true, false>,
                           (const void *)stage_fused2d_kernel<1, false, true>, (const void *)stage_fused2d_kernel<1, true, true>,
                           (const void *)stage_fused2d_kernel<2, false, true>, (const void *)stage_fused2d_kernel<2, true, true> };
    for (const void *f : fns)
        if ((e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FusedSmem<16>::BYTES)) != cudaSuccess)
            return e;
    int nsm = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int ntile = (g.ny + 15) / 16;
    int lz = lz_req > 0 ? lz_req : fused2d_choose_lz(g, nsm);
    if (lz > ntile) lz = ntile;
    p.ty = 16; p.lz = lz;
    p.grid = dim3((g.nx + FTX - 1) / FTX, (ntile + lz - 1) / lz, 1);
    p.base[0] = A; p.base[1] = B;
    for (int b = 0; b < 2; ++b)
        if (!tma::make_state_map(&p.map[b], p.base[b], g.px, g.ny + 2 * NG, 1, g.sy, g.sv, FTX + 4, 16 + 4))
            return cudaErrorNotSupported;
    p.ready = 1;
    return cudaSuccess;
}

template <int STAGE>
inline cudaError_t launch_stage_fused2d(const FusedPlan &p, const Grid &g, const double *in, const double *old,
                                        double *out, double r, const StepScalars *dev_dt, double dx,
                                        StepScalars *red, int inbc, int wrap, cudaStream_t stream)
{
    if (!p.ready) return cudaErrorNotReady;
    const int b = in == p.base[0] ? 0 : 1;
    if (in != p.base[b]) return cudaErrorInvalidValue;
    FusedArgs a;
    a.g = g; a.Uold = old; a.Uout = out; a.dt_over_dx = r; a.dev_dt = dev_dt; a.dx = dx;
    a.red = red; a.lz = p.lz; a.inbc = inbc & 3; a.wrap = wrap; a.zc0 = 0; a.kb = 0; a.km = 0; a.ke = 0; a.nprim = 0; a.lzr = 1;
    const dim3 tb(FTX, 16);
    const size_t smem = FusedSmem<16>::BYTES;
    const bool aniso = g.ry != 1.0;
    if (wrap) {
        if (aniso) stage_fused2d_kernel<STAGE, true, true><<<p.grid, tb, smem, stream>>>(p.map[b], a);
        else       stage_fused2d_kernel<STAGE, false, true><<<p.grid, tb, smem, stream>>>(p.map[b], a);
    } else {
        if (aniso) stage_fused2d_kernel<STAGE, true, false><<<p.grid, tb, smem, stream>>>(p.map[b], a);
        else       stage_fused2d_kernel<STAGE, false, false><<<p.grid, tb, smem, stream>>>(p.map[b], a);
    }
    return cudaGetLastError();
}

}  // namespace hyd
