// hydro_kernels.cuh -- sm_100a kernels of the RK2 Euler step: ghost fill (A1), stage kernels
// (A2-A7), CFL reduction (A8), time-step bookkeeping.  See DESIGN.md section 5 for the layout and
// section 6 for each kernel's roofline.
#pragma once
#include "hydro_faces.cuh"

namespace hyd {

// Padded SoA state (A0): U[v][K][J][I], I fastest, row pitch `px` doubles (multiple of 16),
// active cells I in [2, nx+1] etc.  `lead` doubles precede element (0,0,0) of every variable so
// that the first active cell of every row sits on a 128-byte boundary.
struct Grid {
    int nx, ny, nz;          // active cells (1 on an inactive axis of a 1D / 2D run)
    int px;                  // row pitch (doubles)
    long long sy;            // plane stride = px * (ny + 2 oy)
    long long sv;            // variable stride (doubles), multiple of 16
    int bc[6];
    double gamma, gm1, igm1, theta;
    int ndim;                // active axes: x | x,y | x,y,z  (R21)
    int oy, oz;              // ghost layers per side in y and z: NG on an active axis, 0 otherwise (x: always NG)
    double ry, rz;           // dx/dy, dx/dz: exactly 1 for cubic cells (R23)
};

__device__ __forceinline__ long long cell(const Grid &g, int I, int J, int K)
{
    return (long long)I + (long long)g.px * J + g.sy * K;
}

// element (I, J, K) = first active cell of the padded arrays
__device__ __forceinline__ long long cell0(const Grid &g, int i, int j, int k)
{
    return cell(g, i + NG, j + g.oy, k + g.oz);
}

// Device-resident time step (hydro_run_steps, hydro_evolve): dt = (cfl/ndim) * (dmin / smax), clipped to
// land on t_final exactly (O8 / R14); once t_final is reached further steps get dt = 0, which the
// stage kernels turn into the identity (U + (-(0*D)) = U, 0.5*((U+U)+(-0)) = U, bit for bit).
struct StepScalars {
    unsigned long long smax_bits;   // running max of the CFL reduction (bit pattern)
    int flag;                       // sticky: unphysical state seen
    int done;                       // t has reached t_final
    double dt;                      // time step of the current step
    double t;                       // simulation time (device copy)
    long long steps;                // steps taken since begin_run
    double t_final;                 // +inf for hydro_run_steps
};

__global__ void begin_run_kernel(StepScalars *s, double t0, double t_final)
{
    s->t = t0;
    s->steps = 0;
    s->t_final = t_final;
    s->done = 0;
}

// `cfl_n` = CFL / ndim (formed on the host: one rounding), `dmin` = smallest edge of the cell (R22).
__device__ __forceinline__ void advance_dt(StepScalars *s, double cfl_n, double dmin)
{
    if (s->done) { s->dt = 0.0; return; }
    const double smax = __longlong_as_double((long long)s->smax_bits);
    const double c3 = cfl_n;
    const double dxs = dmin / smax;
    double dt = __dmul_rn(c3, dxs);                    // never contracted: same roundings on every build
    const double t = s->t;
    if (__dadd_rn(t, dt) >= s->t_final) {
        dt = s->t_final - t;
        s->t = s->t_final;
        s->done = 1;
    } else {
        s->t = __dadd_rn(t, dt);
    }
    s->dt = dt;
    s->steps += 1;
}

// Start of a step when no ghost fill is launched (every boundary is handled inside the stage
// kernels): form this step's dt (device-dt steps) and clear the max-signal-speed accumulator for the
// reduction fused into stage 2.  With a ghost fill in the step the same two jobs ride on it.
__global__ void begin_step_kernel(StepScalars *s, int advance, double cfl_n, double dmin)
{
    if (advance) advance_dt(s, cfl_n, dmin);
    s->smax_bits = 0ull;
}

// ------------------------------------------------------------------------------------------
// A1 ghost fill (R9).  One thread per (face pair of one axis, transverse active cell); each
// thread fills the 2+2 ghost cells of its line for all 5 variables.  The three axes are
// independent because only active transverse indices are filled.
// Thread 0 optionally clears the max-signal-speed accumulator for the stage that follows.
// ------------------------------------------------------------------------------------------
__global__ void ghost_fill_kernel(Grid g, double *__restrict__ U,
                                  unsigned long long *__restrict__ clear_smax,
                                  StepScalars *advance, double cfl_n, double dmin, int axes)
{
    // first fill of a device-dt step: one thread also forms this step's dt (the stage kernels that
    // read it are launched after this kernel)
    if (advance && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) advance_dt(advance, cfl_n, dmin);
    // 32-bit index arithmetic (the three face counts are < 2^31 for any grid that fits the device)
    // `axes`: bit a set = fill the ghost layers of axis a (the others are handled elsewhere)
    const unsigned nxy = (axes & 4) ? (unsigned)g.nx * g.ny : 0u, nyz = (axes & 1) ? (unsigned)g.ny * g.nz : 0u,
                   nzx = (axes & 2) ? (unsigned)g.nz * g.nx : 0u;
    unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t == 0 && blockIdx.y == 0 && clear_smax) *clear_smax = 0ull;
    int axis, n;
    long long base, stride;
    if (t < nxy) {                       // z faces: thread per (i,j), coalesced in i
        const int i = (int)(t % (unsigned)g.nx), j = (int)(t / (unsigned)g.nx);
        axis = 2; n = g.nz; base = cell(g, i + NG, j + g.oy, 0); stride = g.sy;
    } else if ((t -= nxy) < nzx) {       // y faces: thread per (i,k), coalesced in i
        const int i = (int)(t % (unsigned)g.nx), k = (int)(t / (unsigned)g.nx);
        axis = 1; n = g.ny; base = cell(g, i + NG, 0, k + g.oz); stride = g.px;
    } else if ((t -= nzx) < nyz) {       // x faces: thread per (j,k)
        const int j = (int)(t % (unsigned)g.ny), k = (int)(t / (unsigned)g.ny);
        axis = 0; n = g.nx; base = cell(g, 0, j + g.oy, k + g.oz); stride = 1;
    } else {
        return;
    }
    const int lo = g.bc[2 * axis], hi = g.bc[2 * axis + 1];
    // x faces, fast path: the two ghost cells of a side are half of a 32-byte sector; storing the
    // whole sector (the other half is row padding nobody reads) spares the DRAM a read-modify-write,
    // and 16-byte vector accesses halve the instruction count.  Needs the sectors to line up
    // (nx % 4 == 0; the first active cell of a row is 128-byte aligned) and >= 2 pad cells per row.
    // One conserved variable per grid row (gridDim.y = 5): five times the threads, and one
    // load -> store round trip per thread instead of a chain of five (the kernel is latency-bound).
    // Splitting further, per side, was slower (52 us vs 37 us at 256^3).
    const int v = blockIdx.y;
    if (axis == 0 && (g.nx & 3) == 0 && g.px - (g.nx + 2 * NG) >= 2) {
        {
            double *a = U + v * g.sv + base;
            const double sgn = (v == 1) ? -1.0 : 1.0;
            const double2 l2 = *reinterpret_cast<const double2 *>(a + 2);       // cells 2, 3
            const double2 h2 = *reinterpret_cast<const double2 *>(a + n);       // cells n, n+1
            double2 gl, gh;
            if (lo == 0)      { gl.x = l2.x; gl.y = l2.x; }
            else if (lo == 1) { gl.x = sgn * l2.y; gl.y = sgn * l2.x; }
            else              { gl = h2; }                   // (x is never a slab interface)
            if (hi == 0)      { gh.x = h2.y; gh.y = h2.y; }
            else if (hi == 1) { gh.x = sgn * h2.y; gh.y = sgn * h2.x; }
            else              { gh = l2; }
            double2 *pl = reinterpret_cast<double2 *>(a - 2), *ph = reinterpret_cast<double2 *>(a + n + 2);
            pl[0] = make_double2(0.0, 0.0); pl[1] = gl;
            ph[0] = gh; ph[1] = make_double2(0.0, 0.0);
        }
        return;
    }
    {
        double *a = U + v * g.sv + base;
        const double sgn = (v == 1 + axis) ? -1.0 : 1.0;
        // sources are always active cells [2, n+1]
        const double a2 = a[2 * stride], a3 = a[3 * stride];
        const double an = a[(long long)n * stride], an1 = a[(long long)(n + 1) * stride];
        double g0, g1, g2, g3;
        if (lo == 0)      { g0 = a2; g1 = a2; }
        else if (lo == 1) { g0 = sgn * a3; g1 = sgn * a2; }
        else              { g0 = an; g1 = an1; }
        if (hi == 0)      { g2 = an1; g3 = an1; }
        else if (hi == 1) { g2 = sgn * an1; g3 = sgn * an; }
        else              { g2 = a2; g3 = a3; }
        // kind 3 (neighbouring slab, z only): those ghost layers belong to the halo exchange
        if (lo != 3) { a[0] = g0; a[stride] = g1; }
        if (hi != 3) { a[(long long)(n + 2) * stride] = g2; a[(long long)(n + 3) * stride] = g3; }
    }
}

// ------------------------------------------------------------------------------------------
// A8 stand-alone CFL reduction: smax = max over active cells of |v| + c_s (O7), as an integer
// atomicMax on the bit pattern (non-negative doubles order like their bit patterns), plus a
// sticky flag for unphysical cells (R12).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_max_to_global(double s, int bad,
                                                    unsigned long long *smax_bits, int *flag)
{
    // NaN never wins a '>' comparison; it is reported through `bad` instead
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double other = __shfl_xor_sync(0xffffffffu, s, o);
        s = other > s ? other : s;
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    __shared__ double wmax[32];
    __shared__ int wbad[32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int lane = tid & 31, wid = tid >> 5;
    const int nw = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
    if (lane == 0) { wmax[wid] = s; wbad[wid] = bad; }
    __syncthreads();
    if (wid == 0) {
        s = lane < nw ? wmax[lane] : 0.0;
        bad = lane < nw ? wbad[lane] : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double other = __shfl_xor_sync(0xffffffffu, s, o);
            s = other > s ? other : s;
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (lane == 0) {
            if (s > 0.0) atomicMax(smax_bits, (unsigned long long)__double_as_longlong(s));
            if (bad) atomicOr(flag, 1);
        }
    }
}

__device__ __forceinline__ double cell_signal_speed(double rho, double mx, double my, double mz,
                                                    double E, double gamma, double gm1, int &bad)
{
    double inv, q;
    const Prim w = primitive(rho, mx, my, mz, E, gm1, inv, q);
    const double s = signal_speed(w, inv, q, gamma);
    if (!(rho > 0.0) || !(w.p > 0.0) || !(s <= 1.79769313486231570e308)) bad = 1;
    return s;
}

__global__ void __launch_bounds__(256)
cfl_reduce_kernel(Grid g, const double *__restrict__ U, unsigned long long *smax_bits, int *flag)
{
    double s = 0.0;
    int bad = 0;
    const long long nrow = (long long)g.ny * g.nz;
    // one warp per x-row at a time: coalesced, grid-stride over rows
    const int lane = threadIdx.x & 31;
    const long long wglobal = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long row = wglobal; row < nrow; row += nwarps) {
        const int j = (int)(row % g.ny), k = (int)(row / g.ny);
        const double *u = U + cell0(g, 0, j, k);
        for (int i = lane; i < g.nx; i += 32) {
            const double c = cell_signal_speed(u[i], u[g.sv + i], u[2 * g.sv + i], u[3 * g.sv + i],
                                               u[4 * g.sv + i], g.gamma, g.gm1, bad);
            s = c > s ? c : s;
        }
    }
    block_max_to_global(s, bad, smax_bits, flag);
}

// ------------------------------------------------------------------------------------------
// Stage kernel, variant 0 ("simple"): one thread per active cell, global loads through L1/L2,
// every slope and face the cell needs recomputed by the thread itself (13-cell stencil).
// Same arithmetic as the fused kernel; kept as the bring-up and cross-check implementation.
// STAGE 1: out = U0 + dU(U0).   STAGE 2: out = 0.5*((U0 + U1) + dU(U1)) (+ fused CFL max).
// ------------------------------------------------------------------------------------------
// flux difference F(i+1/2) - F(i-1/2) along D of one cell, (rho, mx, my, mz, E) order
template <int D>
__device__ __forceinline__ void flux_difference(const Grid &g, const double *__restrict__ U,
                                                long long c, long long stride, double dF[5])
{
    double W[5][5];                         // primitives (rho, vx, vy, vz, p) of cells i-2 .. i+2 along D
#pragma unroll
    for (int o = 0; o < 5; ++o) {
        const long long cc = c + (o - 2) * stride;
        const double Uc[5] = { __ldg(U + cc), __ldg(U + g.sv + cc), __ldg(U + 2 * g.sv + cc),
                               __ldg(U + 3 * g.sv + cc), __ldg(U + 4 * g.sv + cc) };
        HYD_PRIM5(Uc, g.gm1, W[o]);
    }
    double Im[5], Om[5], I0[5], O0[5], Ip[5], Op[5];    // inner / outer face values of cells i-1, i, i+1
    HYD_LIMITED_FACES(g.theta, W[0], W[1], W[2], Im, Om);
    HYD_LIMITED_FACES(g.theta, W[1], W[2], W[3], I0, O0);
    HYD_LIMITED_FACES(g.theta, W[2], W[3], W[4], Ip, Op);
    double Fm[5], Fp[5];
    face_flux<D>(Om, I0, g.gamma, g.igm1, Fm);          // face i-1/2: left = outer(i-1), right = inner(i)
    face_flux<D>(O0, Ip, g.gamma, g.igm1, Fp);          // face i+1/2
#pragma unroll
    for (int v = 0; v < 5; ++v) dF[v] = Fp[v] - Fm[v];
}

template <int STAGE, int NDIM>
__global__ void __launch_bounds__(128)
stage_simple_kernel(Grid g, const double *__restrict__ Uin, const double *Uold, double *Uout,
                    double dt_over_dx, const StepScalars *__restrict__ dev_dt, double dx,
                    StepScalars *__restrict__ red, int kz0)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z + kz0;
    double s = 0.0;
    int bad = 0;
    if (i < g.nx && j < g.ny) {
        const double r = dev_dt ? dev_dt->dt / dx : dt_over_dx;
        const long long c = cell0(g, i, j, k);
        // flux differences of the active dimensions only (R21); those of y and z scaled by dx/dy and
        // dx/dz (R23; exactly 1 for cubic cells)
        double dFx[5], dFy[5], dFz[5];
        flux_difference<0>(g, Uin, c, 1, dFx);
        if (NDIM >= 2) flux_difference<1>(g, Uin, c, g.px, dFy);
        if (NDIM >= 3) flux_difference<2>(g, Uin, c, g.sy, dFz);
        double un[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            double D = dFx[v];
            if (NDIM == 2) {
                const double ty = g.ry * dFy[v];
                D = D + ty;
            } else if (NDIM == 3) {
                const double ty = g.ry * dFy[v];
                const double tz = g.rz * dFz[v];
                D = sum3(D, ty, tz);
            }
            const double dU = -(r * D);
            if (STAGE == 1) {
                un[v] = Uin[v * g.sv + c] + dU;
            } else {
                const double sum = Uold[v * g.sv + c] + Uin[v * g.sv + c];
                un[v] = 0.5 * (sum + dU);
            }
            Uout[v * g.sv + c] = un[v];
        }
        if (STAGE == 2 && red) {
#ifdef HYDRO_VERIFY
            s = cell_signal_speed(un[0], un[1], un[2], un[3], un[4], g.gamma, g.gm1, bad);
#else
            s = fast::signal_speed(un, g.gamma, g.gm1, bad);
            if (!(s <= 1.79769313486231570e308)) { bad = 1; s = 0.0; }      // inf or NaN
#endif
        }
    }
    if (STAGE == 2 && red) block_max_to_global(s, bad, &red->smax_bits, &red->flag);
}

// ------------------------------------------------------------------------------------------
// Slab decomposition along z (the paper's domain decomposition): the two
// active planes next to an interface go to the neighbouring slab's two ghost planes after every
// substep.  MODE 0: padded planes K0, K0+1 -> packed buffer [5][2][ny][nx] (send side);
// MODE 1: packed buffer -> padded planes (receive side); MODE 2: padded planes K0, K0+1 of this
// slab -> padded planes Kd, Kd+1 of the neighbour's state `peer` (same nx, ny, pitch), i.e. the
// exchange as direct peer stores -- over NVLink when `peer` lives on another GPU.
// ------------------------------------------------------------------------------------------
template <int MODE>
__global__ void halo_kernel(Grid g, double *U, double *other, int K0, int Kd, long long peer_sv)
{
    const long long per_var = 2ll * g.ny * g.nx, total = NVAR * per_var;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const int v = (int)(t / per_var);
        const long long r = t % per_var;
        const int i = (int)(r % g.nx);
        const int j = (int)((r / g.nx) % g.ny), l = (int)(r / ((long long)g.nx * g.ny));
        const long long c = v * g.sv + cell(g, i + NG, j + g.oy, K0 + l);
        if (MODE == 0) other[t] = U[c];
        else if (MODE == 1) U[c] = other[t];
        else other[v * peer_sv + cell(g, i + NG, j + g.oy, Kd + l)] = U[c];
    }
}

// ------------------------------------------------------------------------------------------
// pack / unpack between the packed [5][nz][ny][nx] layout and the padded state (device side;
// host pointers go through cudaMemcpy3D in the API layer).
// ------------------------------------------------------------------------------------------
// The library may hold a 3D run with its axes relabelled (hydro_api.cu, "axis order"): the caller's axis a is
// the internal axis ax[a], the caller's variable v the internal variable var[v] (the momentum components
// follow their axes).  n = the caller's extents.  Identity for every other handle.
struct AxisMap {
    int n[3];
    int ax[3];
    int var[NVAR];
};

template <bool TO_PADDED>
__global__ void repack_kernel(Grid g, AxisMap m, double *padded, double *packed, unsigned fields)
{
    const long long nact = (long long)m.n[0] * m.n[1] * m.n[2];
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < nact;
         t += (long long)gridDim.x * blockDim.x) {
        const int iu = (int)(t % m.n[0]);
        const long long jk = t / m.n[0];
        const int ju = (int)(jk % m.n[1]), ku = (int)(jk / m.n[1]);
        const int i = m.ax[0] == 0 ? iu : (m.ax[1] == 0 ? ju : ku);
        const int j = m.ax[0] == 1 ? iu : (m.ax[1] == 1 ? ju : ku);
        const int k = m.ax[0] == 2 ? iu : (m.ax[1] == 2 ? ju : ku);
        const long long c = cell0(g, i, j, k);
#pragma unroll
        for (int v = 0; v < NVAR; ++v) {
            if (!(fields >> v & 1u)) continue;               // selected fields only
            if (TO_PADDED) padded[m.var[v] * g.sv + c] = packed[v * nact + t];
            else packed[v * nact + t] = padded[m.var[v] * g.sv + c];
        }
    }
}

}  // namespace hyd
