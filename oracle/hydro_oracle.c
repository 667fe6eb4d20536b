/*
 * hydro_oracle.c -- CPU fp64 ORACLE for the RK2 step of the 3D compressible-Euler
 * finite-volume update (GenASiS RiemannProblem, arXiv 1812.07977).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_1812_07977_b200/csrc/.
 *
 * What it follows
 * ---------------
 * Control structure: Algorithm 1 "Fluid Evolution", one routine per
 * line of the algorithm, each a whole-grid loop nest over explicitly indexed arrays with an
 * OpenMP `parallel do` on the outer loops -- the paper's own CPU variant (PAPER.md:122-128,
 * 140).  One StorageForm-like block of contiguous columns per intermediate (FluidCurrent,
 * FluidOld, Primitive, Differences, Reconstruction, Fluxes, FluidUpdate),
 * rank-3 indexing with two ghost layers, x fastest.
 * Numerics: the paper prints none (no limiter, solver, EOS or time-step formula), so they
 * are BASELINE.json:north_star's list (primitive recovery, generalized-minmod PLM, HLL,
 * flux divergence, RK2 combine, CFL reduction) under the readings R1-R20 of DESIGN.md
 * section 3 (= SURVEY.md section 8(c)); every routine below names the O-step it implements.
 *
 * Arithmetic: IEEE binary64, one rounding per written operation, in the association
 * written here.  Build with `-O2 -ffp-contract=off` and never -ffast-math (see Makefile);
 * min/max are explicit comparisons so their behaviour is defined by this file.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): P1 uniform state bit-exact, P2 Sod
 * L1 convergence to the exact Riemann solution, P3 periodic conservation to roundoff,
 * P4 bitwise cubic-group symmetry, P5 hand-expanded single-cell update, P6 limiter special
 * cases, P7 HLL closed forms, P8 bitwise translation invariance, P9 wall = mirror,
 * P10 axis relabelling, P11 first dt of config 0.  No function here is "parity unpinned".
 *
 * 1D / 2D runs and non-cubic cells (the
 * RiemannProblem is "an extension of the classic 1D Sod shock tube ... to 2D and 3D"), readings
 * R21-R24 of DESIGN.md: a run of dimension ndim has its first ndim axes active; an inactive
 * axis has one cell, no ghost layers, no ghost exchange and no differences, reconstruction or
 * fluxes (all five variables are still carried); cell edges (dx,dy,dz); the update is
 * -(dt/dx) * [dFx (+ (dx/dy) dFy (+ (dx/dz) dFz))] and the time step (CFL/ndim) * min_d(dx_d) /
 * max(|v|+c_s).  With ndim = 3 and dx = dy = dz every operation reduces to the one above bit for
 * bit (dx/dy = 1 exactly).  Pins: N1 digests of the 3D path before the extension, N2 true-1D Sod
 * L1 convergence, N3 2D x<->y symmetry bitwise, N4 2D = 3D run of z-uniform data at equal dt,
 * N5 1D = 2D run of y-uniform data, N6 anisotropic cells: hand-expanded cell update and
 * relabelling of unequal axes, N7 dt formula values (tests/test_oracle_nd.py).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { BC_OUTFLOW = 0, BC_REFLECT = 1, BC_PERIODIC = 2 };
enum { OK = 0, ERR_ARG = 1, ERR_ALLOC = 2, ERR_UNPHYSICAL = 4, ERR_NOSTATE = 5 };
enum { NVAR = 5, NG = 2 };
/* conserved columns: 0 rho, 1 m_x, 2 m_y, 3 m_z, 4 E ; primitive: 0 rho, 1..3 v, 4 p */

typedef struct oracle_hydro {
    int ndim;                 /* active axes: x (1), x,y (2), x,y,z (3) */
    int nx, ny, nz;           /* active cells (1 on an inactive axis) */
    int gx, gy, gz;           /* ghost layers per side: NG on an active axis, 0 otherwise */
    int Nx, Ny, Nz;           /* padded = active + 2*ghost */
    long ncell;               /* padded cells per column */
    double gamma, gm1, igm1, theta, dx, cfl;
    double dxyz[3];           /* cell edges; dx == dxyz[0] */
    int bc[6];                /* xlo,xhi,ylo,yhi,zlo,zhi */
    double t;
    long long step;
    int have_state;
    /* one contiguous block per StorageForm, column v at Value + v*ncell */
    double *FluidCurrent, *FluidOld, *Primitive, *Differences, *ReconInner, *ReconOuter,
           *Fluxes, *FluxDifference /* 3 dims x NVAR columns */, *FluidUpdate;
} oracle_hydro_t;

static inline double dmin(double a, double b) { return a < b ? a : b; }
static inline double dmax(double a, double b) { return a > b ? a : b; }

/* R17: permutation-symmetric 3-term sum: sort, then (smallest + largest) + middle. */
double oracle_sum3(double a, double b, double c)
{
    double lo = dmin(a, b), hi = dmax(a, b);
    double s0 = dmin(lo, c), s2 = dmax(hi, c);
    double s1 = dmax(lo, dmin(hi, c));
    double t = s0 + s2;
    return t + s1;
}

/* O3 / R4: generalized minmod slope from backward difference a and forward difference b. */
double oracle_minmod(double theta, double a, double b)
{
    double ta = theta * fabs(a);
    double tb = theta * fabs(b);
    double ab = a + b;
    double tc = 0.5 * fabs(ab);
    double m = dmin(dmin(ta, tb), tc);
    if (a > 0.0 && b > 0.0) return m;
    if (a < 0.0 && b < 0.0) return -m;
    return 0.0;
}

/* O2: conserved -> primitive for one cell. */
void oracle_primitive(double gamma, const double U[5], double W[5])
{
    double gm1 = gamma - 1.0;
    double inv = 1.0 / U[0];
    double vx = U[1] * inv, vy = U[2] * inv, vz = U[3] * inv;
    double q = oracle_sum3(vx * vx, vy * vy, vz * vz);
    double hr = 0.5 * U[0];
    double ke = hr * q;
    double ei = U[4] - ke;
    W[0] = U[0]; W[1] = vx; W[2] = vy; W[3] = vz; W[4] = gm1 * ei;
}

/* O4: HLL flux through a face whose normal is axis d (0,1,2) from primitive L/R states. */
static void side_state(double gamma, double igm1, int d, const double W[5],
                       double U[5], double F[5], double *vn_out, double *c_out)
{
    double rho = W[0], p = W[4];
    double vn = W[1 + d];
    double vt1 = W[1 + (d + 1) % 3], vt2 = W[1 + (d + 2) % 3];
    double gp = gamma * p;
    double c2 = gp / rho;
    double c = sqrt(c2);
    double tt = vt1 * vt1 + vt2 * vt2;
    double k = vn * vn + tt;
    double hr = 0.5 * rho;
    double E = p * igm1 + hr * k;
    U[0] = rho; U[1] = rho * W[1]; U[2] = rho * W[2]; U[3] = rho * W[3]; U[4] = E;
    F[0] = U[1 + d];
    F[1] = U[1] * vn; F[2] = U[2] * vn; F[3] = U[3] * vn;
    F[1 + d] = F[1 + d] + p;
    F[4] = (E + p) * vn;
    *vn_out = vn; *c_out = c;
}

void oracle_hll_flux(double gamma, int d, const double WL[5], const double WR[5], double F[5])
{
    double gm1 = gamma - 1.0, igm1 = 1.0 / gm1;
    double UL[5], UR[5], FL[5], FR[5], vL, vR, cL, cR;
    side_state(gamma, igm1, d, WL, UL, FL, &vL, &cL);
    side_state(gamma, igm1, d, WR, UR, FR, &vR, &cR);
    double ap = dmax(0.0, dmax(vL + cL, vR + cR));
    double am = dmax(0.0, dmax(cL - vL, cR - vR));
    double w = 1.0 / (ap + am);
    double pi = ap * am;
    for (int v = 0; v < NVAR; ++v) {
        double num = (ap * FL[v] + am * FR[v]) - pi * (UR[v] - UL[v]);
        F[v] = num * w;
    }
}

/* ------------------------------------------------------------------ handle */

/* Initialize for a run of dimension ndim (R21): n[a] >= 2 and d[a] > 0 on the
 * active axes a < ndim, n[a] == 1 on the others (their d[a] and bc entries are ignored). */
int oracle_create_nd(int ndim, const int n[3], const double d[3], double gamma, const int bc[6],
                     oracle_hydro_t **out)
{
    if (!out || !bc || !n || !d) return ERR_ARG;
    *out = NULL;
    if (ndim < 1 || ndim > 3 || !(gamma > 1.0) || !isfinite(gamma)) return ERR_ARG;
    for (int a = 0; a < 3; ++a) {
        if (a < ndim) {
            if (n[a] < 2 || !(d[a] > 0.0) || !isfinite(d[a])) return ERR_ARG;
            if (bc[2 * a] < 0 || bc[2 * a] > 2 || bc[2 * a + 1] < 0 || bc[2 * a + 1] > 2) return ERR_ARG;
            if ((bc[2 * a] == BC_PERIODIC) != (bc[2 * a + 1] == BC_PERIODIC)) return ERR_ARG;
        } else if (n[a] != 1) return ERR_ARG;
    }
    oracle_hydro_t *h = (oracle_hydro_t *)calloc(1, sizeof *h);
    if (!h) return ERR_ALLOC;
    h->ndim = ndim;
    h->nx = n[0]; h->ny = n[1]; h->nz = n[2];
    h->gx = NG; h->gy = ndim >= 2 ? NG : 0; h->gz = ndim >= 3 ? NG : 0;
    h->Nx = h->nx + 2 * h->gx; h->Ny = h->ny + 2 * h->gy; h->Nz = h->nz + 2 * h->gz;
    h->ncell = (long)h->Nx * h->Ny * h->Nz;
    h->gamma = gamma; h->gm1 = gamma - 1.0; h->igm1 = 1.0 / h->gm1;
    h->theta = 1.4; h->cfl = 0.7;
    for (int a = 0; a < 3; ++a) h->dxyz[a] = a < ndim ? d[a] : d[0];
    h->dx = d[0];
    memcpy(h->bc, bc, sizeof h->bc);
    size_t col = (size_t)h->ncell * sizeof(double);
    double **blocks[] = { &h->FluidCurrent, &h->FluidOld, &h->Primitive, &h->Differences,
                          &h->ReconInner, &h->ReconOuter, &h->Fluxes, &h->FluidUpdate };
    for (unsigned b = 0; b < sizeof blocks / sizeof *blocks; ++b) {
        *blocks[b] = (double *)calloc(NVAR, col);
        if (!*blocks[b]) goto fail;
    }
    h->FluxDifference = (double *)calloc(3 * NVAR, col);
    if (!h->FluxDifference) goto fail;
    *out = h;
    return OK;
fail:
    free(h->FluidCurrent); free(h->FluidOld); free(h->Primitive); free(h->Differences);
    free(h->ReconInner); free(h->ReconOuter); free(h->Fluxes); free(h->FluidUpdate);
    free(h->FluxDifference); free(h);
    return ERR_ALLOC;
}

/* The 3D run with cubic cells of edge dx (R13). */
int oracle_create(int nx, int ny, int nz, double gamma, double dx, const int bc[6],
                  oracle_hydro_t **out)
{
    const int n[3] = { nx, ny, nz };
    const double d[3] = { dx, dx, dx };
    if (out) *out = NULL;
    if (nx < 2 || ny < 2 || nz < 2) return ERR_ARG;
    return oracle_create_nd(3, n, d, gamma, bc, out);
}

int oracle_destroy(oracle_hydro_t *h)
{
    if (!h) return ERR_ARG;
    free(h->FluidCurrent); free(h->FluidOld); free(h->Primitive); free(h->Differences);
    free(h->ReconInner); free(h->ReconOuter); free(h->Fluxes); free(h->FluidUpdate);
    free(h->FluxDifference); free(h);
    return OK;
}

int oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n < 1) return ERR_ARG;
    omp_set_num_threads(n);
    return OK;
#else
    return n == 1 ? OK : ERR_ARG;
#endif
}

int oracle_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int oracle_set_cfl(oracle_hydro_t *h, double cfl)
{
    if (!h || !(cfl > 0.0) || !isfinite(cfl)) return ERR_ARG;
    h->cfl = cfl; return OK;
}

int oracle_set_limiter_theta(oracle_hydro_t *h, double theta)
{
    if (!h || !(theta >= 1.0 && theta <= 2.0)) return ERR_ARG;
    h->theta = theta; return OK;
}

int oracle_get_time(oracle_hydro_t *h, double *t, long long *step)
{
    if (!h) return ERR_ARG;
    if (t) *t = h->t;
    if (step) *step = h->step;
    return OK;
}

#define IDX(h, I, J, K) ((long)(I) + (long)(h)->Nx * ((long)(J) + (long)(h)->Ny * (long)(K)))

/* U packed [5][nz][ny][nx], x fastest, active cells only (Initialize). */
int oracle_set_state(oracle_hydro_t *h, const double *U)
{
    if (!h || !U) return ERR_ARG;
    long nact = (long)h->nx * h->ny * h->nz;
    for (int v = 0; v < NVAR; ++v) {
        double *col = h->FluidCurrent + v * h->ncell;
        for (long c = 0; c < h->ncell; ++c) col[c] = 0.0;
        for (int k = 0; k < h->nz; ++k)
            for (int j = 0; j < h->ny; ++j)
                for (int i = 0; i < h->nx; ++i)
                    col[IDX(h, i + h->gx, j + h->gy, k + h->gz)] =
                        U[v * nact + ((long)k * h->ny + j) * h->nx + i];
    }
    h->t = 0.0; h->step = 0; h->have_state = 1;
    return OK;
}

int oracle_get_state(oracle_hydro_t *h, double *U)
{
    if (!h || !U) return ERR_ARG;
    if (!h->have_state) return ERR_NOSTATE;
    long nact = (long)h->nx * h->ny * h->nz;
    for (int v = 0; v < NVAR; ++v) {
        const double *col = h->FluidCurrent + v * h->ncell;
        for (int k = 0; k < h->nz; ++k)
            for (int j = 0; j < h->ny; ++j)
                for (int i = 0; i < h->nx; ++i)
                    U[v * nact + ((long)k * h->ny + j) * h->nx + i] =
                        col[IDX(h, i + h->gx, j + h->gy, k + h->gz)];
    }
    return OK;
}

/* Test hook: the padded FluidCurrent block [5][Nz][Ny][Nx] as it stands. */
int oracle_get_padded(oracle_hydro_t *h, double *Upad)
{
    if (!h || !Upad) return ERR_ARG;
    memcpy(Upad, h->FluidCurrent, (size_t)NVAR * h->ncell * sizeof(double));
    return OK;
}

/* ------------------------------------------------------------------ O1 GhostExchange */

/* Single domain: GhostExchange reduces to the physical boundary
 * rule (R9).  Axis a, active transverse indices only (edges/corners are never read:
 * the difference loops run j=1..nY, k=1..nZ). */
static void ghost_axis(oracle_hydro_t *h, double *Value, int a)
{
    const int n[3] = { h->nx, h->ny, h->nz };
    const int g[3] = { h->gx, h->gy, h->gz };
    const long s[3] = { 1, h->Nx, (long)h->Nx * h->Ny };
    const int t1 = (a + 1) % 3, t2 = (a + 2) % 3;
    const int na = n[a];
    for (int v = 0; v < NVAR; ++v) {
        double *col = Value + v * h->ncell;
        const double sgn = (v == 1 + a) ? -1.0 : 1.0;   /* normal momentum flips at a wall */
        for (int q2 = g[t2]; q2 < n[t2] + g[t2]; ++q2)
            for (int q1 = g[t1]; q1 < n[t1] + g[t1]; ++q1) {
                double *row = col + q1 * s[t1] + q2 * s[t2];
#define A(I) row[(long)(I) * s[a]]
                switch (h->bc[2 * a]) {              /* low side: ghosts 0,1 */
                case BC_OUTFLOW:  A(0) = A(2); A(1) = A(2); break;
                case BC_REFLECT:  A(1) = sgn * A(2); A(0) = sgn * A(3); break;
                case BC_PERIODIC: A(0) = A(na); A(1) = A(na + 1); break;
                }
                switch (h->bc[2 * a + 1]) {          /* high side: ghosts n+2, n+3 */
                case BC_OUTFLOW:  A(na + 2) = A(na + 1); A(na + 3) = A(na + 1); break;
                case BC_REFLECT:  A(na + 2) = sgn * A(na + 1); A(na + 3) = sgn * A(na); break;
                case BC_PERIODIC: A(na + 2) = A(2); A(na + 3) = A(3); break;
                }
#undef A
            }
    }
}

static void GhostExchange(oracle_hydro_t *h, double *Value)
{
    for (int a = 0; a < h->ndim; ++a) ghost_axis(h, Value, a);      /* active axes only (R21) */
}

/* Test hook: run GhostExchange on FluidCurrent. */
int oracle_ghost_fill(oracle_hydro_t *h)
{
    if (!h) return ERR_ARG;
    if (!h->have_state) return ERR_NOSTATE;
    GhostExchange(h, h->FluidCurrent);
    return OK;
}

/* ------------------------------------------------------------------ kernels of a substep */

/* O2 (R18): primitives of every cell a stencil reads = active cells plus the two-deep
 * face slabs (not edges/corners).  Computed on the whole padded box minus nothing would
 * touch uninitialised corners, so walk the union of the three slabs explicitly. */
static void ComputePrimitive(oracle_hydro_t *h, const double *Value)
{
    const long nc = h->ncell;
    double *P = h->Primitive;
#pragma omp parallel for collapse(2) schedule(static)
    for (int K = 0; K < h->Nz; ++K)
        for (int J = 0; J < h->Ny; ++J) {
            int gK = (K < h->gz || K >= h->nz + h->gz), gJ = (J < h->gy || J >= h->ny + h->gy);
            for (int I = 0; I < h->Nx; ++I) {
                int gI = (I < h->gx || I >= h->nx + h->gx);
                if (gK + gJ + gI > 1) continue;            /* edge / corner: never read */
                long c = IDX(h, I, J, K);
                double U[5], W[5];
                for (int v = 0; v < NVAR; ++v) U[v] = Value[v * nc + c];
                oracle_primitive(h->gamma, U, W);
                for (int v = 0; v < NVAR; ++v) P[v * nc + c] = W[v];
            }
        }
}

/* Loop bounds shared by the per-dimension kernels: along axis d the padded index runs
 * lo..hi (inclusive); the other two axes run over active cells only. */
#define DIM_LOOP_BEGIN(h, d, lo, hi)                                                   \
    {                                                                                  \
        int lo_[3] = { (h)->gx, (h)->gy, (h)->gz };                                    \
        int hi_[3] = { (h)->nx + (h)->gx - 1, (h)->ny + (h)->gy - 1, (h)->nz + (h)->gz - 1 }; \
        lo_[d] = (lo); hi_[d] = (hi);                                                  \
        _Pragma("omp parallel for collapse(2) schedule(static)")                       \
        for (int K = lo_[2]; K <= hi_[2]; ++K)                                         \
            for (int J = lo_[1]; J <= hi_[1]; ++J)                                     \
                for (int I = lo_[0]; I <= hi_[0]; ++I) {                               \
                    const long c = IDX(h, I, J, K);
#define DIM_LOOP_END }}

/* ComputeDifferences (Listing 2, R3):
 * dV(i) = V(i) - V(i-1), paper i = 0..n+2  <=>  padded index 1..n+3. */
static void ComputeDifferences(oracle_hydro_t *h, int d)
{
    const long nc = h->ncell;
    const long s[3] = { 1, h->Nx, (long)h->Nx * h->Ny };
    const int n[3] = { h->nx, h->ny, h->nz };
    const double *V = h->Primitive;
    double *dV = h->Differences;
    DIM_LOOP_BEGIN(h, d, 1, n[d] + 3)
        for (int v = 0; v < NVAR; ++v)
            dV[v * nc + c] = V[v * nc + c] - V[v * nc + c - s[d]];
    DIM_LOOP_END
}

/* ComputeReconstruction (O3): limited slope and inner/outer face values on
 * padded cells 1..n+2 along d. */
static void ComputeReconstruction(oracle_hydro_t *h, int d)
{
    const long nc = h->ncell;
    const long s[3] = { 1, h->Nx, (long)h->Nx * h->Ny };
    const int n[3] = { h->nx, h->ny, h->nz };
    const double *V = h->Primitive, *dV = h->Differences;
    double *Vin = h->ReconInner, *Vout = h->ReconOuter;
    const double theta = h->theta;
    DIM_LOOP_BEGIN(h, d, 1, n[d] + 2)
        for (int v = 0; v < NVAR; ++v) {
            double a = dV[v * nc + c], b = dV[v * nc + c + s[d]];
            double sigma = oracle_minmod(theta, a, b);
            double half = 0.5 * sigma;
            Vin[v * nc + c] = V[v * nc + c] - half;
            Vout[v * nc + c] = V[v * nc + c] + half;
        }
    DIM_LOOP_END
}

/* ComputeFluxes ("RiemannSolverInput" PAPER.md:351; O4): face I+1/2 for padded
 * I = 1..n+1 along d, stored at I; left state = outer(I), right state = inner(I+1). */
static void ComputeFluxes(oracle_hydro_t *h, int d)
{
    const long nc = h->ncell;
    const long s[3] = { 1, h->Nx, (long)h->Nx * h->Ny };
    const int n[3] = { h->nx, h->ny, h->nz };
    const double *Vin = h->ReconInner, *Vout = h->ReconOuter;
    double *F = h->Fluxes;
    const double gamma = h->gamma, igm1 = h->igm1;
    DIM_LOOP_BEGIN(h, d, 1, n[d] + 1)
        double WL[5], WR[5], UL[5], UR[5], FL[5], FR[5], vL, vR, cL, cR;
        for (int v = 0; v < NVAR; ++v) { WL[v] = Vout[v * nc + c]; WR[v] = Vin[v * nc + c + s[d]]; }
        side_state(gamma, igm1, d, WL, UL, FL, &vL, &cL);
        side_state(gamma, igm1, d, WR, UR, FR, &vR, &cR);
        double ap = dmax(0.0, dmax(vL + cL, vR + cR));
        double am = dmax(0.0, dmax(cL - vL, cR - vR));
        double w = 1.0 / (ap + am);
        double pi = ap * am;
        for (int v = 0; v < NVAR; ++v) {
            double num = (ap * FL[v] + am * FR[v]) - pi * (UR[v] - UL[v]);
            F[v * nc + c] = num * w;
        }
    DIM_LOOP_END
}

/* First half of ComputeUpdate (O5): per-dimension flux difference on active cells. */
static void ComputeFluxDifference(oracle_hydro_t *h, int d)
{
    const long nc = h->ncell;
    const long s[3] = { 1, h->Nx, (long)h->Nx * h->Ny };
    const int n[3] = { h->nx, h->ny, h->nz };
    const double *F = h->Fluxes;
    double *dF = h->FluxDifference + (long)d * NVAR * nc;
    DIM_LOOP_BEGIN(h, d, NG, n[d] + NG - 1)
        for (int v = 0; v < NVAR; ++v)
            dF[v * nc + c] = F[v * nc + c] - F[v * nc + c - s[d]];
    DIM_LOOP_END
}

/* ComputeUpdate(TimeStep) -> FluidUpdate (O5 / R23): -(dt/dx) times the sum over
 * the active dimensions of the flux differences, those of y and z scaled by dx/dy and dx/dz
 * (exactly 1 for cubic cells).  Three dimensions: sum3; two: a plain sum; one: the x term. */
static void ComputeUpdate(oracle_hydro_t *h, double dt)
{
    const long nc = h->ncell;
    const double r = dt / h->dx;
    const double ry = h->dx / h->dxyz[1], rz = h->dx / h->dxyz[2];
    const int ndim = h->ndim;
    const double *dFx = h->FluxDifference, *dFy = dFx + NVAR * nc, *dFz = dFy + NVAR * nc;
    double *dU = h->FluidUpdate;
    DIM_LOOP_BEGIN(h, 0, NG, h->nx + NG - 1)
        for (int v = 0; v < NVAR; ++v) {
            double D = dFx[v * nc + c];
            if (ndim == 2) {
                double ty = ry * dFy[v * nc + c];
                D = D + ty;
            } else if (ndim == 3) {
                double ty = ry * dFy[v * nc + c];
                double tz = rz * dFz[v * nc + c];
                D = oracle_sum3(D, ty, tz);
            }
            dU[v * nc + c] = -(r * D);
        }
    DIM_LOOP_END
}

/* Lines 8-11 / 16-19 of Algorithm 1, preceded by the
 * primitive recovery north_star names (R18). */
static void Substep(oracle_hydro_t *h, double dt)
{
    ComputePrimitive(h, h->FluidCurrent);
    for (int d = 0; d < h->ndim; ++d) {
        ComputeDifferences(h, d);
        ComputeReconstruction(h, d);
        ComputeFluxes(h, d);
        ComputeFluxDifference(h, d);
    }
    ComputeUpdate(h, dt);
}

/* One RK2 step, Algorithm 1 lines 6-21, O6. */
int oracle_step(oracle_hydro_t *h, double dt)
{
    if (!h || !(dt > 0.0) || !isfinite(dt)) return ERR_ARG;
    if (!h->have_state) return ERR_NOSTATE;
    const long nc = h->ncell;
    double *Cur = h->FluidCurrent, *Old = h->FluidOld, *Upd = h->FluidUpdate;

    GhostExchange(h, Cur);                        /* line 2 / line 21 of the previous step */
    memcpy(Old, Cur, (size_t)NVAR * nc * sizeof(double));      /* FluidOld = FluidCurrent */

    Substep(h, dt);
    DIM_LOOP_BEGIN(h, 0, NG, h->nx + NG - 1)      /* FluidCurrent = FluidOld + FluidUpdate */
        for (int v = 0; v < NVAR; ++v)
            Cur[v * nc + c] = Old[v * nc + c] + Upd[v * nc + c];
    DIM_LOOP_END

    GhostExchange(h, Cur);                        /* line 14 */

    Substep(h, dt);
    DIM_LOOP_BEGIN(h, 0, NG, h->nx + NG - 1)      /* 0.5*(FluidOld+FluidCurrent+FluidUpdate) */
        for (int v = 0; v < NVAR; ++v) {
            double s = Old[v * nc + c] + Cur[v * nc + c];
            double w = s + Upd[v * nc + c];
            Cur[v * nc + c] = 0.5 * w;
        }
    DIM_LOOP_END

    h->t = h->t + dt;
    h->step += 1;
    return OK;
}

/* ------------------------------------------------------------------ O7 ComputeTimeStep */

int oracle_max_signal_speed(oracle_hydro_t *h, double *smax_out)
{
    if (!h || !smax_out) return ERR_ARG;
    if (!h->have_state) return ERR_NOSTATE;
    const long nc = h->ncell;
    const double *Cur = h->FluidCurrent;
    double smax = 0.0;
    int bad = 0;
#pragma omp parallel for collapse(2) schedule(static) reduction(max : smax) reduction(| : bad)
    for (int K = h->gz; K < h->nz + h->gz; ++K)
        for (int J = h->gy; J < h->ny + h->gy; ++J)
            for (int I = h->gx; I < h->nx + h->gx; ++I) {
                long c = IDX(h, I, J, K);
                double rho = Cur[c], mx = Cur[nc + c], my = Cur[2 * nc + c],
                       mz = Cur[3 * nc + c], E = Cur[4 * nc + c];
                double inv = 1.0 / rho;
                double vx = mx * inv, vy = my * inv, vz = mz * inv;
                double q = oracle_sum3(vx * vx, vy * vy, vz * vz);
                double hr = 0.5 * rho;
                double ke = hr * q;
                double ei = E - ke;
                double p = h->gm1 * ei;
                double gp = h->gamma * p;
                double c2 = gp * inv;
                double s = sqrt(q) + sqrt(c2);
                if (!(rho > 0.0) || !(p > 0.0) || !isfinite(s)) bad |= 1;
                if (s > smax) smax = s;
            }
    *smax_out = smax;
    return bad ? ERR_UNPHYSICAL : OK;
}

/* dt = (CFL/ndim) * (min_d dx_d / smax)   (R8 / R22: Courant factor divided by the number of
 * unsplit dimensions, smallest edge of the cell). */
int oracle_cfl_dt(oracle_hydro_t *h, double *dt)
{
    if (!h || !dt) return ERR_ARG;
    double smax;
    int rc = oracle_max_signal_speed(h, &smax);
    if (rc != OK) return rc;
    double dmin_ = h->dxyz[0];
    for (int a = 1; a < h->ndim; ++a) dmin_ = dmin(dmin_, h->dxyz[a]);
    double c3 = h->cfl / (double)h->ndim;
    double dxs = dmin_ / smax;
    *dt = c3 * dxs;
    return OK;
}

/* O8: Algorithm 1 lines 3-4 and 23, with the last step clipped to land on t_final (R14). */
int oracle_evolve(oracle_hydro_t *h, double t_final, long long *nsteps)
{
    if (!h || !isfinite(t_final)) return ERR_ARG;
    if (!h->have_state) return ERR_NOSTATE;
    if (t_final < h->t) return ERR_ARG;
    long long n = 0;
    while (h->t < t_final) {
        double dt;
        int rc = oracle_cfl_dt(h, &dt);
        if (rc != OK) return rc;
        int last = 0;
        if (h->t + dt >= t_final) { dt = t_final - h->t; last = 1; }
        rc = oracle_step(h, dt);
        if (rc != OK) return rc;
        if (last) h->t = t_final;
        ++n;
    }
    if (nsteps) *nsteps = n;
    return OK;
}
