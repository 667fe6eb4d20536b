// hydro_stage_fused.cuh -- the fused RK-stage kernel (A2-A8 of DESIGN.md section 2) for sm_100a.
//
// One launch per Runge-Kutta substep does primitive recovery, the three per-dimension limited
// reconstructions, the HLL face fluxes, the flux divergence, the stage combination and (stage 2)
// the max-signal-speed reduction, i.e. the paper's ComputeDifferences / ComputeReconstruction /
// ComputeFluxes / ComputeUpdate and the "FluidCurrent = ..." lines of Algorithm 1
// without any of its intermediate storages.
//
// Shape.  The kernel is not bound by HBM (each value crosses it once per stage) but by
// how well fp64 work, shared-memory exchange and the TMA stream overlap at 16 warps per SM, so the design
// minimises fp64 instructions per cell: every slope and every face flux is computed exactly once.
//   * A block owns a TX x TY column tile (x fastest, one warp per x-row of 32 cells) and marches
//     along z over a chunk of `lz` planes.  A thread owns the column (i, j).
//   * z direction: a register pipeline.  When plane kk arrives the thread has W(kk-2), W(kk-1),
//     computes W(kk), the z-slope of cell kk-1 and the flux through face (kk-2)+1/2, which
//     completes cell kk-2.  Nothing in z is ever recomputed or exchanged.
//   * x and y directions of plane kk-2: primitives of (tile + 2-cell plus-shaped halo) go to
//     shared memory once; each thread computes the slopes of its own cell, hands its outer face
//     value to the +x / +y neighbour through shared memory, computes the flux through its low
//     face and hands that to the -x / -y neighbour's divergence.  The tile's extra high-edge
//     faces and the two halo-cell slopes they need are a flattened list whose owner rotates over
//     the warps from plane to plane.
//   * the conserved planes (tile + halo, all five variables) arrive through a TMA ring
//     (cp.async.bulk.tensor, one 4-D box per plane); the three hand-offs per plane are split-phase
//     mbarriers with z-direction work between arrive and wait (see the kernel).
//   * conserved state crosses HBM once per stage (interior planes; halos and the four extra
//     planes per chunk re-read through L2).
#pragma once
#include "hydro_kernels.cuh"
#include "hydro_tma.cuh"

namespace hyd {

constexpr int FTX = 32;            // tile width: one warp per row

constexpr int FNS = 4;             // TMA ring depth: planes kk-2, kk-1, kk resident + kk+1 in flight

// Shared-memory carve-up (doubles).  The ring stages and the primitive tile share one layout,
// [v][row][col] with pitch WP -- the layout the TMA box arrives in.
template <int TY> struct FusedSmem {
    static constexpr int WP = FTX + 4;                 // pitch of a (tile + halo) plane
    static constexpr int WROWS = TY + 4;
    static constexpr int WSZ = WROWS * WP;             // per variable
    static constexpr int STAGE = NVAR * WSZ;           // one ring stage (multiple of 16 doubles)
    static constexpr int XP = FTX + 2;                 // pitch of x-face arrays (FTX+1 used)
    static constexpr int XSZ = TY * XP;
    static constexpr int YSZ = (TY + 1) * FTX;
    static constexpr int OFF_RING = 0;                 // raw conserved planes, filled by TMA
    static constexpr int OFF_W = OFF_RING + FNS * STAGE;  // primitives of the plane being updated
    static constexpr int NW = TY == 16 ? 2 : 1;        // primitive tiles (2: by plane parity, no W barrier)
    static constexpr int OFF_OX = OFF_W + NW * STAGE;  // outer x-face value of cell i-1 at slot i;
    static constexpr int OFF_FX = OFF_OX;              //   overwritten in place by the flux through i-1/2
    static constexpr int OFF_OY = OFF_OX + NVAR * XSZ; // outer y-face value of row j-1 at row j;
    static constexpr int OFF_FY = OFF_OY;              //   overwritten in place by the flux through j-1/2
    static constexpr int OFF_IXE = OFF_OY + NVAR * YSZ; // inner x-face value of cell i0+TX, per row
    static constexpr int OFF_IYE = OFF_IXE + NVAR * TY; // inner y-face value of row j0+TY, per col
    static constexpr int OFF_OXE = OFF_IYE + NVAR * FTX; // outer x-face value of cell i0+TX-1, per row, x2 (plane parity)
    static constexpr int OFF_BAR = OFF_OXE + 2 * NVAR * TY; // FNS TMA mbarriers + 3 phase mbarriers
    static constexpr int TOTAL = OFF_BAR + FNS + 3 + 1;
    static constexpr size_t BYTES = (size_t)TOTAL * sizeof(double);
    static constexpr unsigned STAGE_BYTES = STAGE * sizeof(double);
    static_assert(STAGE_BYTES % 128 == 0, "TMA destination stages must stay 128-byte aligned");
};

}  // namespace hyd

#include "hydro_stage_fused_kernel.cuh"
