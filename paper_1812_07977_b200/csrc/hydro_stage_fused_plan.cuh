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
    cudaError_t e = cudaFuncSetAttribute(stage_fused_kernel<STAGE, TY, MINB, false>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)FusedSmem<TY>::BYTES);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(stage_fused_kernel<STAGE, TY, MINB, true>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FusedSmem<TY>::BYTES);
}

inline void fused_geometry(FusedPlan &p, const Grid &g, int ty, int lz)
{
    p.ty = ty;
    p.lz = lz < 1 ? 1 : (lz > g.nz ? g.nz : lz);
    p.grid = dim3((g.nx + FTX - 1) / FTX, (g.ny + ty - 1) / ty, (g.nz + p.lz - 1) / p.lz);
}

// Planes per chunk: fill whole waves of (SMs x resident blocks) as evenly as possible while
// keeping the four extra planes a chunk streams (two below, two above) a small overhead.
inline int fused_choose_lz(const Grid &g, int ty, int nsm, int per_sm)
{
    const long long tiles = (long long)((g.nx + FTX - 1) / FTX) * ((g.ny + ty - 1) / ty);
    const long long slots = (long long)nsm * per_sm;
    int best = g.nz;
    double best_cost = 1e300;
    for (int l = g.nz < 4 ? g.nz : 4; l <= g.nz; ++l) {
        const long long blocks = tiles * ((g.nz + l - 1) / l);
        const long long waves = (blocks + slots - 1) / slots;
        const double cost = (double)waves * (l + 4);          // time ~ waves x planes per block
        if (cost < best_cost - 1e-9) { best_cost = cost; best = l; }
    }
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
    // 32 x 16 tiles (one 512-thread block per SM) carry half the per-warp halo / edge work of 32 x 8
    // tiles (two 256-thread blocks per SM) and win on large grids (256^3: 1.615 vs 1.636 ms per
    // step); small grids need the finer tiling to fill the machine
    int ty = g.ny >= 128 ? 16 : 8;
    if (ty_req) ty = ty_req == 16 ? 16 : 8;
    int lz = fused_choose_lz(g, ty, nsm, ty == 16 ? 1 : 2);
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
                                      int inbc, cudaStream_t stream)
{
    if (!p.ready) return cudaErrorNotReady;
    const int b = in == p.base[0] ? 0 : 1;
    if (in != p.base[b]) return cudaErrorInvalidValue;
    FusedArgs a;
    a.g = g; a.Uold = old; a.Uout = out; a.dt_over_dx = r; a.dev_dt = dev_dt; a.dx = dx;
    a.red = red; a.lz = p.lz; a.inbc = inbc;
    const bool aniso = g.ry != 1.0 || g.rz != 1.0;            // non-cubic cells: two more DMUL per variable
    if (p.ty == 16) {
        if (aniso) stage_fused_kernel<STAGE, 16, 1, true><<<p.grid, dim3(FTX, 16), FusedSmem<16>::BYTES, stream>>>(p.map[b], a);
        else       stage_fused_kernel<STAGE, 16, 1, false><<<p.grid, dim3(FTX, 16), FusedSmem<16>::BYTES, stream>>>(p.map[b], a);
    } else {
        if (aniso) stage_fused_kernel<STAGE, 8, 2, true><<<p.grid, dim3(FTX, 8), FusedSmem<8>::BYTES, stream>>>(p.map[b], a);
        else       stage_fused_kernel<STAGE, 8, 2, false><<<p.grid, dim3(FTX, 8), FusedSmem<8>::BYTES, stream>>>(p.map[b], a);
    }
    return cudaGetLastError();
}

}  // namespace hyd
