// hydro_stage_fused_plan.cuh -- host side of the fused stage kernel: launch geometry, TMA
// descriptors of the two state buffers, launch.
#pragma once

namespace hyd {

// Cost of a block's start (barrier set-up, first TMA round trip, the four warm-up planes that only cost
// primitives and z-slopes) in plane times: fit to measured whole-column, 64- and 32-plane chunks at
// 32 x 16 (2.98 us per plane and stage, 3.7 us per block).
constexpr double FUSED_WARM = 1.25;
constexpr int FUSED_SLAB_UNIT = 16;   // balanced layers: planes next to a slab interface that are computed first

// z partition of one launch over the active planes [kb, ke): chunks of lz planes over [kb, km) and,
// when km < ke, thinner chunks of lzr planes over the remainder [km, ke)
struct FusedLayers {
    int kb = -1, ke = -1;            // the range this partition was made for (cache key)
    int lz = 0, km = 0, nprim = 0;   // chunks of lz planes over [kb, km): layers 0 .. nprim-1
    int lzr = 1, nlayer = 0;         // chunks of lzr planes over [km, ke): layers nprim .. nlayer-1
    double cost = 0.0;
};

struct FusedPlan {
    int ready = 0;
    int ty = 8;              // tile height (8: two blocks per SM, 16: one)
    int lz = 32;             // 3D: planes per z-chunk of a whole-domain launch; 2D: tile rows per chunk
    int km = 0;              // 3D: whole-domain launch: chunks cover [0, km), thinner remainder layers [km, nz)
    int lz_req = 0;          // 3D: the caller's planes per chunk (0: choose per launch range)
    int nsm = 148;
    FusedLayers part[4];     // 3D: partitions of the plane ranges launched so far ([0]: the whole domain)
    int npart = 0;
    dim3 grid;               // grid of a whole-domain launch
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

inline long long fused_tiles(const Grid &g, int ty)
{
    return (long long)((g.nx + FTX - 1) / FTX) * ((g.ny + ty - 1) / ty);
}

// Uniform chunks.  A chunk of l planes takes about (l + FUSED_WARM) plane times; blocks are handed to the
// SMs in waves of (SMs x resident blocks).  Measured on B200 (tiling sweep): the
// best uniform chunking is the one that fills whole waves, short chunks are cheap, 32 x 16 tiles (one
// block per SM) beat 32 x 8 tiles (two per SM) at equal wave count because they carry half the halo work,
// and a lone 32 x 8 block on an SM runs about 1.5 times faster than when it shares the SM (tiny grids:
// more, smaller blocks win).
inline double fused_cost(const Grid &g, int ty, int nzr, int l, int nsm)
{
    const long long blocks = fused_tiles(g, ty) * ((nzr + l - 1) / l);
    const int per_sm = ty == 16 ? 1 : 2;
    const long long slots = (long long)nsm * per_sm;
    const long long waves = (blocks + slots - 1) / slots;
    double cost = (double)waves * (l + FUSED_WARM);
    if (ty == 8 && blocks <= nsm) cost *= 0.65;              // one 8-warp block per SM
    if (ty == 16) cost *= 0.92;                              // half the halo / edge work per cell
    return cost;
}

inline int fused_choose_lz(const Grid &g, int ty, int nzr, int nsm, double *cost_out = nullptr)
{
    int best = nzr;
    double best_cost = 1e300;
    for (int l = nzr; l >= (nzr < 2 ? nzr : 2); --l) {           // ties: the longer chunk (fewer blocks)
        const double cost = fused_cost(g, ty, nzr, l, nsm);
        if (cost < best_cost - 1e-9) { best_cost = cost; best = l; }
    }
    if (cost_out) *cost_out = best_cost;
    return best;
}

// Balanced layers: with T tiles and S resident slots (T <= S), q = S / T primary layers of m / q planes
// put one block on each of q T slots; the planes [m, nzr) left over form a remainder of p thin layers
// whose p T blocks run on the other L = S - q T slots in ceil(p T / L) rounds.  m balances the two:
//     m / q + w = rounds ((nzr - m) / p + w),      w = FUSED_WARM plane times of warm-up per block.
// Every slot then streams about nzr T / S planes whatever the grid's extents; the blocks of a layer sweep
// z in lockstep, so neighbouring tiles share their halo columns in L2 as with uniform chunks.
inline bool fused_balanced_layers(const Grid &g, int ty, int kb, int ke, int nsm, FusedLayers &out)
{
    const int nzr = ke - kb;
    const long long T = fused_tiles(g, ty), S = (long long)nsm * (ty == 16 ? 1 : 2);
    if (T > S || nzr < 4) return false;
    const long long q = S / T, L = S - q * T;
    if (q > nzr / 2) return false;                                // tiny grids: uniform short chunks
    const double w = FUSED_WARM;
    int m = nzr, pieces = 0;
    double best = (double)((nzr + q - 1) / q) + w;                // no remainder: q equal layers
    for (int p = 1; L > 0 && p <= 4; ++p) {
        const long long rounds = (T * p + L - 1) / L;
        auto both = [&](int mm) {
            const double a = (double)((mm + q - 1) / q) + w, b = (double)rounds * ((nzr - mm + p - 1) / p + w);
            return a > b ? a : b;
        };
        const int m0 = (int)((rounds * (nzr / (double)p + w) - w) / (1.0 / q + rounds / (double)p));
        for (int mm = m0 - 2; mm <= m0 + 2; ++mm)                 // integer planes: take the best neighbour
            if (mm >= 2 * q && mm <= nzr - 2 * p && both(mm) < best - 1e-9) { best = both(mm); m = mm; pieces = p; }
    }
    out.lz = (int)((m + q - 1) / q);
    out.km = kb + m;
    out.nprim = (m + out.lz - 1) / out.lz;
    out.lzr = pieces ? (nzr - m + pieces - 1) / pieces : 1;
    out.nlayer = out.nprim + (pieces ? (nzr - m + out.lzr - 1) / out.lzr : 0);
    out.cost = best * (ty == 16 ? 0.92 : 1.0);
    return true;
}

// The partition of one launch: the caller's chunk length if given, else the cheaper of the best uniform
// chunking and the balanced layers.
inline FusedLayers fused_partition(const Grid &g, int ty, int kb, int ke, int nsm, int lz_req)
{
    FusedLayers u;
    const int nzr = ke - kb;
    u.km = ke; u.lzr = 1;
    if (lz_req > 0) u.lz = lz_req > nzr ? nzr : lz_req, u.cost = fused_cost(g, ty, nzr, u.lz, nsm);
    else u.lz = fused_choose_lz(g, ty, nzr, nsm, &u.cost);
    u.nprim = u.nlayer = (nzr + u.lz - 1) / u.lz;
    if (lz_req > 0) return u;
    FusedLayers b;
    if (fused_balanced_layers(g, ty, kb, ke, nsm, b) && b.cost < u.cost) return b;
    return u;
}

inline dim3 fused_grid(const Grid &g, int ty, int nzr, const FusedLayers &z)
{
    return dim3((g.nx + FTX - 1) / FTX, (g.ny + ty - 1) / ty, z.nlayer);
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
    const FusedLayers z8 = fused_partition(g, 8, 0, g.nz, nsm, lz_req), z16 = fused_partition(g, 16, 0, g.nz, nsm, lz_req);
    int ty = z16.cost <= z8.cost ? 16 : 8;
    if (ty_req) ty = ty_req == 16 ? 16 : 8;
    const FusedLayers &z = ty == 16 ? z16 : z8;
    p.ty = ty; p.lz = z.lz; p.km = z.km; p.lz_req = lz_req; p.nsm = nsm;
    p.part[0] = z; p.part[0].kb = 0; p.part[0].ke = g.nz; p.npart = 1;
    p.grid = fused_grid(g, ty, g.nz, z);
    p.base[0] = A; p.base[1] = B;
    for (int b = 0; b < 2; ++b)
        if (!tma::make_state_map(&p.map[b], p.base[b], g.px, g.ny + 2 * NG, g.nz + 2 * NG, g.sy, g.sv,
                                 FTX + 4, ty + 4))
            return cudaErrorNotSupported;     // no TMA descriptor -> no fused kernel (fail loudly)
    p.ready = 1;
    return cudaSuccess;
}

template <int STAGE>
inline cudaError_t launch_stage_fused(FusedPlan &p, const Grid &g, const double *in,
                                      const double *old, double *out, double r,
                                      const StepScalars *dev_dt, double dx, StepScalars *red,
                                      int inbc, int wrap, cudaStream_t stream, int kb = 0, int ke = -1)
{
    if (!p.ready) return cudaErrorNotReady;
    const int b = in == p.base[0] ? 0 : 1;
    if (in != p.base[b]) return cudaErrorInvalidValue;
    FusedArgs a;
    a.g = g; a.Uold = old; a.Uout = out; a.dt_over_dx = r; a.dev_dt = dev_dt; a.dx = dx;
    if (ke < 0) ke = g.nz;
    if (ke <= kb) return cudaSuccess;
    // the z partition of this range of planes (slab runs launch the interface planes first)
    int ip = 0;
    while (ip < p.npart && (p.part[ip].kb != kb || p.part[ip].ke != ke)) ++ip;
    if (ip == p.npart) {
        if (p.npart == 4) ip = p.npart = 1;                   // (a slab run uses three ranges)
        p.part[ip] = fused_partition(g, p.ty, kb, ke, p.nsm, p.lz_req);
        p.part[ip].kb = kb; p.part[ip].ke = ke;
        p.npart = ip + 1;
    }
    const FusedLayers &z = p.part[ip];
    a.red = red; a.lz = z.lz; a.inbc = inbc; a.wrap = wrap; a.zc0 = 0;
    a.kb = kb; a.km = z.km; a.ke = ke; a.nprim = z.nprim; a.lzr = z.lzr;
    const dim3 grid = fused_grid(g, p.ty, ke - kb, z);
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
