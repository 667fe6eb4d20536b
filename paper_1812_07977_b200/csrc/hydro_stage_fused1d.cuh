// hydro_stage_fused1d.cuh -- fused RK-stage kernel of 1D runs (the paper's RiemannProblem runs in 1D,
// 2D and 3D; R21: the y and z axes carry one cell, no ghost layers and no
// differences, slopes or fluxes).
//
// A tile is F1T consecutive cells of the single row, one cell per thread.  Primitives of the tile
// and its two-cell halo go to shared memory once; every thread computes the slope of its own cell and
// hands its outer face value to the +x neighbour, computes the HLL flux through its low face over the
// face value it consumed, and takes the flux through its high face from the +x neighbour: each slope
// and each flux once (the simple kernel recomputes a five-cell stencil per thread, 2.6 times the fp64
// work), three block barriers per tile.  With 130 / 171 fp64 instructions against 80 / 120 bytes
// per cell and stage the 1D step is bound by HBM, not by the fp64 pipe: plain coalesced loads with
// many resident blocks keep enough bytes in flight, so there is no TMA ring here: a block walks tiles of
// 128 cells with the next tile's own values fetched one tile ahead, five blocks per SM.  The boundary
// rule of x is applied in the kernel -- a ghost cell is read from its source cell (clamp / mirror / wrap):
// three launches per step, the ghost cells in memory are never touched.  Same building blocks as the
// other stage kernels (hydro_faces.cuh), so the verification build reproduces the oracle bit for bit.
#pragma once
#include "hydro_kernels.cuh"

namespace hyd {

// measured on B200 (2^20 / 2^24 cells, G cell-updates/s): 128 cells x 5 blocks per SM 18.7 / 19.8,
// 128 x 6 17.2 / 19.1 (spills), 128 x 4 18.2 / 18.3, 256 x 3 16.7 / 18.7, 64 x 10 16.0 / 17.7
constexpr int F1T = 128;               // cells per tile, one per thread
constexpr int F1_BLOCKS_PER_SM = 5;

template <int STAGE>
__global__ void __launch_bounds__(F1T, F1_BLOCKS_PER_SM)
stage_fused1d_kernel(Grid g, const double *__restrict__ Uin, const double *Uold, double *Uout,
                     double dt_over_dx, const StepScalars *__restrict__ dev_dt, double dx,
                     StepScalars *__restrict__ red, int inbc)
{
    __shared__ double Ws[NVAR][F1T + 4];     // primitives of cells i0-2 .. i0+F1T+1
    __shared__ double Os[NVAR][F1T + 1];     // slot s: outer face value of cell i0+s-1, overwritten in place
                                             // by the flux through face i0+s-1/2
    __shared__ double Ie[NVAR];              // inner face value of cell i0+F1T
    const int tx = threadIdx.x;
    const long long c0 = cell0(g, 0, 0, 0);
    const double gamma = g.gamma, gm1 = g.gm1, igm1 = g.igm1, theta = g.theta;
    const double r = dev_dt ? dev_dt->dt / dx : dt_over_dx;
    const int ntile = (g.nx + F1T - 1) / F1T;
    // inbc: the boundary rule of x is applied here (a ghost cell takes the state of its source cell: nearest
    // cell / mirror image with the normal momentum negated / periodic image) and the ghost cells in
    // memory are never read; otherwise they are read from memory.  Cells past the high ghost layer
    // are never used by an active cell: clamped to stay addressable.
    auto load_plain = [&](const double *U, int ii, double out[5]) {
        const long long c = c0 + min(ii, g.nx + NG - 1);
#pragma unroll
        for (int v = 0; v < 5; ++v) out[v] = __ldg(U + v * g.sv + c);
    };
    auto load_mapped = [&](const double *U, int ii, double out[5]) {
        bool flip = false;
        const long long c = c0 + bc_source(ii, g.nx, g.bc[0], g.bc[1], 0, g.nx - 1, flip);
#pragma unroll
        for (int v = 0; v < 5; ++v) out[v] = __ldg(U + v * g.sv + c);
        out[1] = flip_sign(out[1], flip);
    };
    // only the first and the last tile hold ghost cells (block-uniform)
    auto edge_tile = [&](int tile) { return inbc && (tile == 0 || (tile + 1) * F1T + NG > g.nx); };
    auto load_cell = [&](bool edge, const double *U, int ii, double out[5]) {
        if (edge) load_mapped(U, ii, out); else load_plain(U, ii, out);
    };
    double s = 0.0;
    int bad = 0;
    // a block walks the tiles blockIdx.x, blockIdx.x + gridDim.x, ...; the own values of the next tile
    // (and stage 2's U0) are fetched before the current tile is computed, so their latency is hidden
    double Un[5], Uon[5];
    if ((int)blockIdx.x < ntile) {
        load_cell(edge_tile(blockIdx.x), Uin, blockIdx.x * F1T + tx, Un);
        if (STAGE == 2) load_plain(Uold, blockIdx.x * F1T + tx, Uon);      // (used by active cells only)
    }
#pragma unroll 1
    for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    const int i0 = tile * F1T, i = i0 + tx;
    const bool active = i < g.nx;
    double Uc[5], Uo[5], Wc[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { Uc[v] = Un[v]; if (STAGE == 2) Uo[v] = Uon[v]; }
    if (tile + (int)gridDim.x < ntile) {
        load_cell(edge_tile(tile + gridDim.x), Uin, i + gridDim.x * F1T, Un);
        if (STAGE == 2) load_plain(Uold, i + gridDim.x * F1T, Uon);
    }
    HYD_PRIM5(Uc, gm1, Wc);
#pragma unroll
    for (int v = 0; v < 5; ++v) Ws[v][tx + 2] = Wc[v];
    if (tx < 4) {                                            // halo cells i0-2, i0-1, i0+F1T, i0+F1T+1
        const int hs = tx < 2 ? tx : F1T + tx;
        double Uh[5], Wh[5];
        load_cell(edge_tile(tile), Uin, i0 - 2 + hs, Uh);
        HYD_PRIM5(Uh, gm1, Wh);
#pragma unroll
        for (int v = 0; v < 5; ++v) Ws[v][hs] = Wh[v];
    }
    __syncthreads();

    double In[5];
    {
        double Wm[5], Wp[5], Ou[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) { Wm[v] = Ws[v][tx + 1]; Wp[v] = Ws[v][tx + 3]; }
        HYD_LIMITED_FACES(theta, Wm, Wc, Wp, In, Ou);
#pragma unroll
        for (int v = 0; v < 5; ++v) Os[v][tx + 1] = Ou[v];
    }
    if (tx < 2) {                                            // the halo cells next to the tile: i0-1 (outer), i0+F1T (inner)
        const int hs = tx == 0 ? 1 : F1T + 2;
        double Wm[5], W0[5], Wp[5], Ih[5], Oh[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) { Wm[v] = Ws[v][hs - 1]; W0[v] = Ws[v][hs]; Wp[v] = Ws[v][hs + 1]; }
        HYD_LIMITED_FACES(theta, Wm, W0, Wp, Ih, Oh);
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            if (tx == 0) Os[v][0] = Oh[v]; else Ie[v] = Ih[v];
        }
    }
    __syncthreads();

    double Fl[5];
    {
        double L[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) L[v] = Os[v][tx];
        face_flux<0>(L, In, gamma, igm1, Fl);
#pragma unroll
        for (int v = 0; v < 5; ++v) Os[v][tx] = Fl[v];
    }
    if (tx == 0) {                                           // the tile's high face
        double L[5], R[5], F[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) { L[v] = Os[v][F1T]; R[v] = Ie[v]; }
        face_flux<0>(L, R, gamma, igm1, F);
#pragma unroll
        for (int v = 0; v < 5; ++v) Os[v][F1T] = F[v];
    }
    __syncthreads();

    if (active) {
        const long long c = c0 + i;
        double un[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double D = Os[v][tx + 1] - Fl[v];          // one active dimension (O5)
            const double dU = -(r * D);
            if (STAGE == 1) {
                un[v] = Uc[v] + dU;
            } else {
                const double sum = Uo[v] + Uc[v];
                un[v] = 0.5 * (sum + dU);
            }
            Uout[v * g.sv + c] = un[v];
        }
        if (STAGE == 2 && red) {
#ifdef HYDRO_VERIFY
            const double sc = cell_signal_speed(un[0], un[1], un[2], un[3], un[4], gamma, gm1, bad);
            s = sc > s ? sc : s;
#else
            s = fast::max_nonneg(s, fast::signal_speed(un, gamma, gm1, bad));
#endif
        }
    }
    __syncthreads();                                         // the tile's shared arrays are free again
    }
#ifndef HYDRO_VERIFY
    if (!(s <= 1.79769313486231570e308)) { bad = 1; s = 0.0; }      // inf or NaN pattern won
#endif
    if (STAGE == 2 && red) block_max_to_global(s, bad, &red->smax_bits, &red->flag);
}

template <int STAGE>
inline cudaError_t launch_stage_fused1d(const Grid &g, const double *in, const double *old, double *out, double r,
                                        const StepScalars *dev_dt, double dx, StepScalars *red, int inbc,
                                        cudaStream_t stream)
{
    int nsm = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int ntile = (g.nx + F1T - 1) / F1T, slots = nsm * F1_BLOCKS_PER_SM;
    stage_fused1d_kernel<STAGE><<<ntile < slots ? ntile : slots, F1T, 0, stream>>>(g, in, old, out, r, dev_dt, dx, red, inbc);
    return cudaGetLastError();
}

}  // namespace hyd
