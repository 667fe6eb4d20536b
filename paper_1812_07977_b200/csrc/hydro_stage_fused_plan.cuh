// hydro_stage_fused_plan.cuh -- host side of the fused stage kernel: launch geometry, TMA
// descriptors of the two state buffers, launch.
#pragma once

namespace hyd {

struct FusedPlan {
    int ready = 0;
    int ty = 8;              // tile height (8: two blocks per SM, 16: one)
    int lz = 32;             // planes per z-chunk
    dim3 grid;
    const double *base[2] = { nullptr, nullptr };   // the two state buffers ...
    CUtensorMap map[2];                              // ... and their TMA descriptors for box (36, ty+4, 1, 5)
};

template <int STAGE, int TY, int MINB>
inline cudaError_t fused_set_attr()
{
    const void *fns[4] = { (const void *)stage_fused_kernel<STAGE, TY, MINB, false, false>,
                           (const void *)stage_fused_kernel<STAGE, TY, MINB, true, false>,
                           (const void *)stage_fused_kernel<STAGE, TY, MINB, false, true>,
                           (const void *)stage_fused_kernel<STAGE, TY, MINB, true, true> };
    for (const void *f : fns) {
        cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FusedSmem<TY>::BYTES);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

inline void fused_geometry(FusedPlan &p, const Grid &g, int ty, int lz)
{
    p.ty = ty;
    p.lz = lz < 1 ? 1 : (lz > g.nz ? g.nz : lz);
    p.grid = dim3((g.nx + FTX - 1) / FTX, (g.ny + ty - 1) / ty, (g.nz + p.lz - 1) / p.lz);
}

// Launch geometry.  A block streams (l + 4) planes for l computed ones, but the four warm-up planes
// only cost primitives and z-slopes, so with the block prologue a chunk of l planes takes about
// (l + 2) plane times; blocks are handed to the SMs in waves of (SMs x resident blocks).  Measured on
// B200 (tiling sweep): the best geometry is the one that fills whole waves,
// short chunks are cheap, 32 x 16 tiles (one block per SM) beat 32 x 8 tiles (two per SM) at equal
// wave count because they carry half the halo work, and a lone 32 x 8 block on an SM runs about 1.5
// times faster than when it shares the SM (tiny grids: more, smaller blocks win).
inline double fused_cost(const Grid &g, int ty, int l, int nsm)
{
    const long long tiles = (long long)((g.nx + FTX - 1) / FTX) * ((g.ny + ty - 1) / ty);
    const long long blocks = tiles * ((g.nz + l - 1) / l);
    const int per_sm = ty == 16 ? 1 : 2;
    const long long slots = (long long)nsm * per_sm;
    const long long waves = (blocks + slots - 1) / slots;
    double cost = (double)waves * (l + 2);
    if (ty == 8 && blocks <= nsm) cost *= 0.65;              // one 8-warp block per SM
    if (ty == 16) cost *= 0.92;                              // half the halo / edge work per cell
    return cost;
}

inline int fused_choose_lz(const Grid &g, int ty, int nsm, double *cost_out = nullptr)
{
    int best = g.nz;
    double best_cost = 1e300;
    for (int l = g.nz; l >= (g.nz < 2 ? g.nz : 2); --l) {       // ties: the longer chunk (fewer blocks)
        const double cost = fused_cost(g, ty, l, nsm);
        if (cost < best_cost - 1e-9) { best_cost = cost; best = l; }
    }
    if (cost_out) *cost_out = best_cost;
    return best;
}

// ty_req / lz_req: 0 = choose (hydro_set_tiling); otherwise the tile height (8 | 16) and the planes
// per z-chunk the caller asked for.
inline cudaError_t plan_stage_fused(FusedPlan &p, const Grid &g, const double *A, const double *B,
                                    int ty_req = 0, int lz_req = 0)
{
    cudaError_t e;
    if ((e = fused_set_attr<1, 16, 1>()) != cudaSuccess) return e;
    if ((e = fused_set_attr<2, 16, 1>()) != cudaSuccess) return e;
    if ((e = fused_set_attr<1, 8, 2>()) != cudaSuccess) return e;
    if ((e = fused_set_attr<2, 8, 2>()) != cudaSuccess) return e;
    int nsm = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess)
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    double c8, c16;
    const int l8 = fused_choose_lz(g, 8, nsm, &c8), l16 = fused_choose_lz(g, 16, nsm, &c16);
    int ty = c16 <= c8 ? 16 : 8;
    if (ty_req) ty = ty_req == 16 ? 16 : 8;
    int lz = ty == 16 ? l16 : l8;
    if (lz_req > 0) lz = lz_req;
    fused_geometry(p, g, ty, lz);
    p.base[0] = A; p.base[1] = B;
    for (int b = 0; b < 2; ++b)
        if (!tma::make_state_map(&p.map[b], p.base[b], g.px, g.ny + 2 * NG, g.nz + 2 * NG, g.sy, g.sv,
                                 FTX + 4, ty + 4))
            return cudaErrorNotSupported;     // no TMA descriptor -> no fused kernel (fail loudly)
    p.ready = 1;
    return cudaSuccess;
}

template <int STAGE>
inline cudaError_t launch_stage_fused(const FusedPlan &p, const Grid &g, const double *in,
                                      const double *old, double *out, double r,
                                      const StepScalars *dev_dt, double dx, StepScalars *red,
                                      int inbc, int wrap, cudaStream_t stream, int zc0 = 0, int nzc = -1)
{
    if (!p.ready) return cudaErrorNotReady;
    const int b = in == p.base[0] ? 0 : 1;
    if (in != p.base[b]) return cudaErrorInvalidValue;
    FusedArgs a;
    a.g = g; a.Uold = old; a.Uout = out; a.dt_over_dx = r; a.dev_dt = dev_dt; a.dx = dx;
    a.red = red; a.lz = p.lz; a.inbc = inbc; a.wrap = wrap; a.zc0 = zc0;
    dim3 grid = p.grid;
    if (nzc >= 0) grid.z = (unsigned)nzc;                     // a range of z-chunks (slab runs: interface chunks first)
    if (grid.z == 0) return cudaSuccess;
    const bool aniso = g.ry != 1.0 || g.rz != 1.0;            // non-cubic cells: two more DMUL per variable
    // template switches keep the common case (cubic cells, no periodic x / y) free of their code
#define HYD_LAUNCH(TYv, MINBv, AN, WR)                                                              \
    stage_fused_kernel<STAGE, TYv, MINBv, AN, WR><<<grid, dim3(FTX, TYv), FusedSmem<TYv>::BYTES, stream>>>(p.map[b], a)
    if (p.ty == 16) {
        if (wrap) { if (aniso) HYD_LAUNCH(16, 1, true, true); else HYD_LAUNCH(16, 1, false, true); }
        else      { if (aniso) HYD_LAUNCH(16, 1, true, false); else HYD_LAUNCH(16, 1, false, false); }
    } else {
        if (wrap) { if (aniso) HYD_LAUNCH(8, 2, true, true); else HYD_LAUNCH(8, 2, false, true); }
        else      { if (aniso) HYD_LAUNCH(8, 2, true, false); else HYD_LAUNCH(8, 2, false, false); }
    }
#undef HYD_LAUNCH
    return cudaGetLastError();
}

}  // namespace hyd
