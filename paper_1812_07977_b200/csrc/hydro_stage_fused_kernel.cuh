// hydro_stage_fused_kernel.cuh -- body of the fused stage kernel (see hydro_stage_fused.cuh).
#pragma once

namespace hyd {

// Layers.  blockIdx.x / .y = tile, blockIdx.z = layer: the planes [kb, km) in chunks of lz planes and,
// when km < ke, the planes [km, ke) in thinner chunks of lzr planes.  Uniform chunking has km = ke; the
// balanced partition (hydro_stage_fused_plan.cuh) makes the chunks of [kb, km) fill the resident slots
// of the device once and hands the remainder to the slots left over.  Neighbouring tiles of a layer
// sweep z in lockstep and share their halo columns in L2.

struct FusedArgs {
    Grid g;
    const double *Uold;     // stage 2: U0 (read at the thread's own cell only); may alias Uout
    double *Uout;
    double dt_over_dx;      // used when dev_dt == nullptr
    const StepScalars *dev_dt;
    double dx;
    StepScalars *red;       // stage 2: max-signal-speed accumulator + sticky flag (or nullptr)
    int lz;                 // planes per z-chunk (2D: tile rows per chunk)
    int zc0;                // 2D kernel only
    int kb, km, ke;         // 3D: this launch updates the active planes [kb, ke): layers blockIdx.z < nprim are the
    int nprim, lzr;         // chunks of lz planes of [kb, km), the others the chunks of lzr planes of [km, ke)
    int wrap;               // bit 0 / 1: x / y is periodic and this kernel maintains its ghost layers: every
                            // updated cell within two cells of such a face is also stored to its ghost image
    int inbc;               // bit a: the boundary rule of axis a is applied by this kernel (ghost layers of
                            // that axis are never read from memory); 0: all ghosts come from memory
};

// Boundary rule of one axis (O1 / R9) as an index map: the active cell whose state a ghost cell
// takes (outflow: nearest active cell; reflecting: mirror image, normal momentum negated; periodic:
// wrap).  i is an active-cell index; only the two ghost layers [-2,-1] and [n, n+1] matter, indices
// further out are never used and are clamped into [cmin, cmax] (the caller's tile) to stay addressable.
// Branch-free: the boundary kinds are uniform, the selects cost a handful of integer instructions.
__device__ __forceinline__ int bc_source(int i, int n, int lo, int hi, int cmin, int cmax, bool &flip)
{
    // kind 3 (neighbouring slab): the ghost layers exist in memory, written by the halo exchange
    const int below = lo == 0 ? 0 : (lo == 1 ? -1 - i : (lo == 2 ? i + n : i));
    const int above = hi == 0 ? n - 1 : (hi == 1 ? 2 * n - 1 - i : (hi == 2 ? i - n : i));
    flip = (i < 0 && lo == 1) || (i >= n && hi == 1);
    const int s = i < 0 ? below : (i >= n ? above : i);
    return min(max(s, cmin), cmax);
}

__device__ __forceinline__ double flip_sign(double x, bool f)
{
    return __hiloint2double(__double2hiint(x) ^ (f ? (int)0x80000000 : 0), __double2loint(x));
}

// `umap` describes the stencil input (stage 1: U0, stage 2: U1) to the TMA unit.
//
// Boundaries (GhostExchange of Algorithm 1).  Axes in `inbc` are handled here:
// z ghost planes are never materialised -- the TMA plane coordinate is remapped to the source plane
// (clamp / mirror / wrap); x and y ghost cells of outflow and reflecting faces are read from their
// source cell inside the tile when the primitives are formed (own-cell source `wsrc` of the threads
// that stand in for ghost cells, index map of the halo cells), with the normal momentum negated at
// a wall.  Periodic x / y ghosts need cells from the far side of the domain, outside the tile's box:
// they stay in memory (those axes are not in `inbc`) and are kept current by the PRODUCER -- the
// update stores every cell within two cells of a periodic face a second time, at its ghost image
// (`wrap`); ghost_fill_kernel only runs once after the state was set from outside.
//
// Synchronisation.  The x/y exchange of one plane needs block-wide hand-offs (primitives, outer
// face values, fluxes).  Each is a split-phase mbarrier: a warp ARRIVES as soon as its stores are
// done, then does work that needs no other warp (the filler), and only then WAITS.  The skew
// between warps is absorbed by the fillers instead of idling at a barrier.
//   TY = 16 (PIPE): the primitive tile is double-buffered by plane parity, so its hand-off rides on
//   the flux barrier, and only the y-slopes (and the halo-cell slopes) precede the face-value
//   barrier -- the x-slopes stay inside the warp (lane i -> lane i+1) and run as filler:
//     per cell plane c:  y-slopes, halo slopes  arrive_O  [x-slopes, prim(c+4), z-slope]  wait_O
//                        tile(c+1), x/y fluxes, edge fluxes  arrive_F  [z-flux]  wait_F  update
//   TY = 8 (two blocks per SM, single primitive tile):
//     per cell plane c:  wait_W  x/y slopes  arrive_O  [prim(c+4), z-slope]  wait_O  fluxes  arrive_F
//                        [z-flux, tile(c+1), arrive_W(c+1)]  wait_F  update
template <int STAGE, int TY, int MINB, bool ANISO, bool WRAP>
__global__ void __launch_bounds__(FTX * TY, MINB)
stage_fused_kernel(const __grid_constant__ CUtensorMap umap, const FusedArgs a)
{
    using S = FusedSmem<TY>;
    constexpr int TX = FTX, WP = S::WP, XP = S::XP;
    extern __shared__ __align__(128) double sm[];
    constexpr bool PIPE = S::NW == 2;      // see "Synchronisation" above
    double *Oxs = sm + S::OFF_OX, *Oys = sm + S::OFF_OY;
    double *Fxs = sm + S::OFF_FX, *Fys = sm + S::OFF_FY;
    double *Ixe = sm + S::OFF_IXE, *Iye = sm + S::OFF_IYE;
    uint64_t *bar = reinterpret_cast<uint64_t *>(sm + S::OFF_BAR);     // TMA: plane p -> bar[p % FNS]
    uint64_t *barW = bar + FNS, *barO = bar + FNS + 1, *barF = bar + FNS + 2;

    const Grid &g = a.g;
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * TX + tx;
    const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;     // tile origin, active coordinates
    const int zl = blockIdx.z, zr = zl - a.nprim;             // chunk = active planes [k0, k1)
    const int k0 = zr < 0 ? a.kb + zl * a.lz : a.km + zr * a.lzr;
    const int k1 = zr < 0 ? min(k0 + a.lz, a.km) : min(k0 + a.lzr, a.ke);
    const int nc = k1 - k0;                                   // cell planes; raw planes 0..nc+3
    const int nplanes = nc + 4;                               //   (raw plane p = active plane k0-2+p)
    const double gamma = g.gamma, gm1 = g.gm1, igm1 = g.igm1, theta = g.theta;
    const long long sv = g.sv;

    // own column; threads past the active range still compute (they own the domain's high-edge
    // faces) but never touch global memory
    const bool active = (i0 + tx < g.nx) && (j0 + ty < g.ny);
    const long long col = (long long)(i0 + tx + NG) + (long long)g.px * (j0 + ty + NG);
    const int wc = (ty + 2) * WP + tx + 2;                    // own cell in a (tile + halo) plane
    // Threads just past the active range stand in for the ghost cells of the domain's high faces:
    // their primitives come from the ghost cell's source cell (in-kernel boundary rule).  Nothing of
    // this is kept in registers: the map is recomputed by those (few, inactive) threads only, and
    // the wall flags of z are block-uniform.
    auto load_own = [&](const double *Ust, int p, double Un[5]) {
        int ws = wc;
        bool fx = false, fy = false;
        if (!active && (a.inbc & 3)) {
            const int is = (a.inbc & 1) ? bc_source(i0 + tx, g.nx, g.bc[0], g.bc[1], i0 - NG, i0 + TX + NG - 1, fx) : i0 + tx;
            const int js = (a.inbc & 2) ? bc_source(j0 + ty, g.ny, g.bc[2], g.bc[3], j0 - NG, j0 + TY + NG - 1, fy) : j0 + ty;
            ws = (js - j0 + NG) * WP + (is - i0 + NG);
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) Un[v] = Ust[v * S::WSZ + ws];
        if (!active) { Un[1] = flip_sign(Un[1], fx); Un[2] = flip_sign(Un[2], fy); }
        if ((a.inbc & 4) && (g.bc[4] == 1 || g.bc[5] == 1)) {  // a wall in z: mirror planes carry -m_z
            const int kz = k0 + p - NG;                        // active z index of the plane
            Un[3] = flip_sign(Un[3], (g.bc[4] == 1 && kz < 0) || (g.bc[5] == 1 && kz >= g.nz));
        }
    };
    // tiles that touch a boundary handled here remap their halo cells (block-uniform)
    const bool edge_tile = ((a.inbc & 1) && (i0 == 0 || i0 + TX + NG > g.nx)) ||
                           ((a.inbc & 2) && (j0 == 0 || j0 + TY + NG > g.ny));

    // The tile's extra work (halo primitives, halo-cell slopes, high-edge faces) is a flattened
    // list handed out by ROLE = (warp + plane) mod TY, so that it rotates over the warps from plane
    // to plane: every warp (and every SM sub-partition, warp % 4) carries the same load over TY
    // planes, and the short-term imbalance stays inside the slack of the split barriers.
    //   roles 0,1: high-edge x / y faces;  roles 2,3: y halo slopes;  role 6: x halo slopes;
    //   roles 3..: halo primitives (x halo on role 3, y halo on the following ones).
    static_assert(TY >= 8 && (TY & (TY - 1)) == 0, "role rotation needs a power-of-two warp count >= 8");
    constexpr int NHX = 4 * TY, NH = 4 * TY + 4 * TX;

    if (t == 0) {
#pragma unroll
        for (int s = 0; s < FNS; ++s) tma::mbar_init(&bar[s], 1);
        tma::mbar_init(barW, TY); tma::mbar_init(barO, TY); tma::mbar_init(barF, TY);
        tma::fence_barrier_init();
    }
    __syncthreads();
    auto request_plane = [&](int p) {                         // thread 0 only
        tma::mbar_arrive_expect_tx(&bar[p % FNS], S::STAGE_BYTES);
        // z ghost planes are never materialised: request the source plane instead (clamp / mirror / wrap)
        bool fz;
        const int K = (a.inbc & 4) ? bc_source(k0 + p - NG, g.nz, g.bc[4], g.bc[5], -NG, g.nz + NG - 1, fz) + NG : k0 + p;
        tma::load_4d(sm + S::OFF_RING + (p % FNS) * S::STAGE, &umap, i0, j0, K, 0, &bar[p % FNS]);
    };
    if (t == 0)
        for (int p = 0; p < FNS; ++p) request_plane(p);       // nplanes >= 5 > FNS

    const double r = a.dev_dt ? a.dev_dt->dt / a.dx : a.dt_over_dx;

    // primitive tile of one cell plane: own cell from registers, halo cells from the raw plane
    auto write_tile = [&](double *Wsm, const double Wown[5], const double *Uraw, int role) {
#pragma unroll
        for (int v = 0; v < 5; ++v) Wsm[v * S::WSZ + wc] = Wown[v];
        const int th = (role - 3) * TX + tx;                  // halo cell index -> plane coords (hc, hr)
        if (th >= 0 && th < NH) {
            int hc, hr;
            if (th < NHX) { const int q = th & 3; hr = (th >> 2) + 2; hc = q < 2 ? q : TX + q; }
            else { const int u = th - NHX, q = u / TX; hc = (u % TX) + 2; hr = q < 2 ? q : TY + q; }
            const int hw = hr * WP + hc;
            int hs = hw;
            bool fx = false, fy = false;
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
        if (!PIPE) {
            __syncwarp();
            if (tx == 0) tma::mbar_arrive(barW);
        }
    };

    // ---- prologue: raw planes 0..3 -> W(k0), W(k0+1), outer_z(k0), flux through face k0-1/2 ----
    double Wa[5], Wb[5];          // W(k), W(k+1) of the current cell plane k
    double Oz[5];                 // outer z-face value of cell k
    double Fzm[5];                // flux through face k-1/2
    double smax = 0.0;
    int bad = 0;
#pragma unroll
    for (int v = 0; v < 5; ++v) { Wa[v] = Wb[v] = Oz[v] = Fzm[v] = 0.0; }
#pragma unroll 1
    for (int p = 0; p < 4; ++p) {
        tma::mbar_wait(&bar[p], 0);
        double Un[5], Wn[5];
        load_own(sm + S::OFF_RING + p * S::STAGE, p, Un);
        HYD_PRIM5(Un, gm1, Wn);
        if (p >= 2) {
            double Iz[5], Ozn[5];
            HYD_LIMITED_FACES(theta, Wa, Wb, Wn, Iz, Ozn);    // cell of raw plane p-1
            if (p == 3) face_flux<2>(Oz, Iz, gamma, igm1, Fzm);
#pragma unroll
            for (int v = 0; v < 5; ++v) Oz[v] = Ozn[v];
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) { Wa[v] = Wb[v]; Wb[v] = Wn[v]; }
        if (p == 1) {                                         // raw plane 0 has been read by everyone
            __syncthreads();
            if (t == 0) { tma::fence_proxy_async(); request_plane(4); }
        }
    }
    write_tile(sm + S::OFF_W, Wa, sm + S::OFF_RING + 2 * S::STAGE, ty);   // cell plane 0 = raw plane 2; arrive_W(0)
    if (PIPE) __syncthreads();

#pragma unroll 1
    for (int c = 0; c < nc; ++c) {
        const uint32_t par = c & 1;
        const int role = (ty + c) & (TY - 1);
        const double *Uk = sm + S::OFF_RING + ((c + 2) % FNS) * S::STAGE;      // raw plane of cell plane c
        const long long cg = col + g.sy * (long long)(k0 + c + NG);
        double *Wsm = sm + S::OFF_W + (PIPE ? (c & 1) * S::STAGE : 0);
        // stage 2 reads its own U0 values with plain loads behind the flux hand-off (no shared memory left to
        // stage them through); their DRAM latency showed up as long-scoreboard stalls on the first use.  Lanes
        // 0..9 of every warp ask L2 for the warp's row of the NEXT plane, one 128-byte line each (variable
        // lane / 2, half lane % 2): one instruction per warp and plane (256^3: stage 2 -3.4 %, 128^3: -3.9 %,
        // 512^3: -4 %; two planes ahead: the same, three: less).
        if (STAGE == 2 && tx < 2 * NVAR && j0 + ty < g.ny && c + 1 < nc) {
            const int v = tx >> 1, half = tx & 1;
            if (half * 16 < g.nx - i0) tma::prefetch_l2_line(a.Uold + v * sv + (cg - tx) + g.sy + half * 16);
        }
        if (!PIPE) tma::mbar_wait(barW, par);
        // ---- P2: x and y slopes of the own cell (W(k) = Wa), outer face values out ----------
        double Ix[5], Iy[5];
        if (!PIPE) {
            double Wm[5], Wp[5], Ox[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wm[v] = Wsm[v * S::WSZ + wc - 1]; Wp[v] = Wsm[v * S::WSZ + wc + 1]; }
            HYD_LIMITED_FACES(theta, Wm, Wa, Wp, Ix, Ox);
#pragma unroll
            for (int v = 0; v < 5; ++v) Oxs[v * S::XSZ + ty * XP + tx + 1] = Ox[v];
        }
        {
            double Wm[5], Wp[5], Oy[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wm[v] = Wsm[v * S::WSZ + wc - WP]; Wp[v] = Wsm[v * S::WSZ + wc + WP]; }
            HYD_LIMITED_FACES(theta, Wm, Wa, Wp, Iy, Oy);
#pragma unroll
            for (int v = 0; v < 5; ++v) Oys[v * S::YSZ + (ty + 1) * TX + tx] = Oy[v];
        }
        // halo-cell slopes: x: cells (-1, j) -> outer, (TX, j) -> inner; y: rows -1 -> outer, TY -> inner
        // (PIPE: the own x-slopes run after arrive_O, so role 7 also forms the outer value of cell
        // TX-1 of every row, which the high-edge x-faces of role 0 read right after wait_O)
        if (role == 2 || role == 3 || (role == 6 && tx < 2 * TY) || (PIPE && role == 7 && tx < TY)) {
            int cc, st, dst, dstride;
            bool want_outer;
            if (role == 6) {
                const int j = tx >> 1, hi = tx & 1;
                cc = (j + 2) * WP + (hi ? TX + 2 : 1); st = 1; want_outer = !hi;
                dst = hi ? S::OFF_IXE + j : S::OFF_OX + j * XP;
                dstride = hi ? TY : S::XSZ;
            } else if (PIPE && role == 7) {
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
        if (PIPE) {   // own x-slopes as filler: the outer values stay inside the warp (lane i -> lane i+1)
            double Wm[5], Wp[5], Ox[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { Wm[v] = Wsm[v * S::WSZ + wc - 1]; Wp[v] = Wsm[v * S::WSZ + wc + 1]; }
            HYD_LIMITED_FACES(theta, Wm, Wa, Wp, Ix, Ox);
            if (tx != TX - 1) {
#pragma unroll
                for (int v = 0; v < 5; ++v) Oxs[v * S::XSZ + ty * XP + tx + 1] = Ox[v];
            }
        }
        // ---- filler O: primitives of raw plane c+4, z-slope of cell plane c+1 ---------------
        double Wn[5], Iz[5], Ozn[5];
        {
            const int p = c + 4;
            tma::mbar_wait(&bar[p % FNS], (p / FNS) & 1);
            double Un[5];
            load_own(sm + S::OFF_RING + (p % FNS) * S::STAGE, p, Un);
            HYD_PRIM5(Un, gm1, Wn);
            HYD_LIMITED_FACES(theta, Wa, Wb, Wn, Iz, Ozn);
        }
        tma::mbar_wait_sync(barO, par);
        if (PIPE) __syncwarp();                               // the warp's own outer x values are in place
        // every warp is past P4 of cell plane c-1: raw plane c+1 is dead, refill its stage
        if (t == 0 && c + 5 < nplanes) { tma::fence_proxy_async(); request_plane(c + 5); }
        // ---- P3: x and y fluxes through the low faces ---------------------------------------
        double Fxl[5], Fyl[5];
        // PIPE: primitive tile of cell plane c+1 into the other buffer (free since wait_F(c-1), read
        // after wait_F(c)); own cell = W(c+1) = Wb, halo cells from raw plane c+3
        if (PIPE && c + 1 < nc)
            write_tile(sm + S::OFF_W + ((c + 1) & 1) * S::STAGE, Wb,
                       sm + S::OFF_RING + ((c + 3) % FNS) * S::STAGE, (ty + c + 1) & (TY - 1));
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
        // the tile's high-edge faces: role 0 lanes < TY: x face of row `lane`; role 1: y face of
        // column `lane` (each flux is written over the outer value it consumed)
        if (role == 0 && tx < TY) {
            double L[5], R[5], F[5];
            const double *Le = PIPE ? sm + S::OFF_OXE + (c & 1) * NVAR * TY + tx : Oxs + tx * XP + TX;
            constexpr int les = PIPE ? TY : S::XSZ;
#pragma unroll
            for (int v = 0; v < 5; ++v) { L[v] = Le[v * les]; R[v] = Ixe[v * TY + tx]; }
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
        // ---- filler F: U0 loads in flight (stage 2) ------------------------------------------
        double Uo[5];
        if (STAGE == 2) {
#pragma unroll
            for (int v = 0; v < 5; ++v) Uo[v] = active ? a.Uold[v * sv + cg] : 0.0;
        }
        // z flux through face k+1/2; rotate the z pipeline; primitive tile of cell plane c+1
        double dFz[5];
        {
            double Fzp[5];
            face_flux<2>(Oz, Iz, gamma, igm1, Fzp);
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                dFz[v] = Fzp[v] - Fzm[v]; Fzm[v] = Fzp[v]; Oz[v] = Ozn[v]; Wa[v] = Wb[v]; Wb[v] = Wn[v];
            }
        }
        if (!PIPE && c + 1 < nc)                            // arrive_W(c+1)
            write_tile(Wsm, Wa, sm + S::OFF_RING + ((c + 3) % FNS) * S::STAGE, (ty + c + 1) & (TY - 1));
        // stage 1: the own conserved values are fetched before the wait (their latency hides behind
        // it; measured -0.8 %); stage 2 has no registers to spare across the wait (+1.7 % there)
        double u1r[5];
        if (STAGE == 1) {
#pragma unroll
            for (int v = 0; v < 5; ++v) u1r[v] = Uk[v * S::WSZ + wc];
        }
        tma::mbar_wait_sync(barF, par);
        // ---- P4: divergence, RK combine, store, CFL ------------------------------------------
        double un[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double dFx = Fxs[v * S::XSZ + ty * XP + tx + 1] - Fxl[v];
            double dFy = Fys[v * S::YSZ + (ty + 1) * TX + tx] - Fyl[v];
            if (ANISO) { dFy = g.ry * dFy; dFz[v] = g.rz * dFz[v]; }    // non-cubic cells (R23): dx/dy, dx/dz
            const double D = HYD_SUM3(dFx, dFy, dFz[v]);
            const double dU = -(r * D);
            const double u1 = STAGE == 1 ? u1r[v] : Uk[v * S::WSZ + wc];
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
    }
    if (STAGE == 2 && a.red) {
        if (!(smax <= 1.79769313486231570e308)) { bad = 1; smax = 0.0; }   // inf or NaN pattern won
        block_max_to_global(smax, bad, &a.red->smax_bits, &a.red->flag);
    }
}

}  // namespace hyd

#include "hydro_stage_fused_plan.cuh"
