/* oracle/pic_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64, single-threaded CPU statement of the particle step that the
 * CUDA library under paper_2110_08650_b200/csrc computes in fp32:
 *     gather (CIC/TSC/PQS) -> relativistic Boris push -> move -> Esirkepov deposit
 *     -> periodic wrap and supercell re-bucket.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call it.  It shares no code, header, table or helper with
 * the CUDA path and is never imported by the product.
 *
 * Source of the definitions.  The paper (§3.1)
 * describes the method in three sentences and names none of the algorithms; they are
 * fixed by BASELINE.json:north_star and written out as the textbook definitions in
 * SURVEY.md §8(c) steps 1-7 (readings S1-S7, S14, S16 — every one "paper silent").
 * Each function below cites the step it follows.  Nothing is blocked, fused, tiled
 * or reordered beyond those definitions; windows are deliberately generous
 * (floor(X)-3 .. floor(X)+4, eight nodes per axis) so that no order-specific index
 * logic exists that could be wrong — a shape function is simply zero outside its
 * support.
 *
 * Units: c = 1, u = gamma*v/c, du/dt = (q/m)(E + v x B).  Positions inside this file
 * are in CELL units (X = x/dx); the grid is periodic on all axes (S6).
 * Parity pins: tests/test_oracle_*.py (moments, closed forms, continuity, six-path
 * brute force, worked examples of SURVEY.md §8(c)).  No function here is "parity
 * unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t nx, ny, nz;      /* grid cells */
    int32_t scx, scy, scz;   /* supercell size in cells */
    int32_t order;           /* 1 CIC, 2 TSC, 3 PQS (polynomial degree, reading S2) */
    int32_t gather;          /* 0 momentum-conserving gather (reading S3, the contract's path); 1 energy-conserving
                              * (Galerkin) gather: order o-1 along every axis a component is staggered on */
    double dx, dy, dz, dt;
} orc_params;

#define ORC_WLO (-3)
#define ORC_WN 8            /* window nodes per axis: floor(X)-3 .. floor(X)+4 */

/* Yee stagger of Ex,Ey,Ez,Bx,By,Bz along x,y,z. */
static const double ORC_STAG[6][3] = {
    {0.5, 0.0, 0.0}, {0.0, 0.5, 0.0}, {0.0, 0.0, 0.5},
    {0.0, 0.5, 0.5}, {0.5, 0.0, 0.5}, {0.5, 0.5, 0.0}};

static int orc_wrap(long i, int n) { long r = i % n; if (r < 0) r += n; return (int)r; }

/* Step 1: B-spline assignment functions W_o(d), d = distance to the node in cells. */
double orc_shape(int order, double d)
{
    double a = fabs(d);
    if (order == 0) return (d >= -0.5 && d < 0.5) ? 1.0 : 0.0;   /* nearest grid point; a particle midway belongs to the upper node */
    if (order == 1) return a < 1.0 ? 1.0 - a : 0.0;
    if (order == 2) {
        if (a <= 0.5) return 0.75 - a * a;
        if (a <= 1.5) { double t = 1.5 - a; return 0.5 * t * t; }
        return 0.0;
    }
    if (order == 3) {
        if (a <= 1.0) return 2.0 / 3.0 - a * a + 0.5 * a * a * a;
        if (a <= 2.0) { double t = 2.0 - a; return t * t * t / 6.0; }
        return 0.0;
    }
    return NAN;
}

/* Step 3: momentum-conserving direct interpolation of one staggered component,
 * F_c(X) = sum_ijk F_c[i,j,k] W(Xx-(i+sx)) W(Xy-(j+sy)) W(Xz-(k+sz)), indices wrapped.
 * F is indexed i + nx*(j + ny*k). */
double orc_gather_component(const orc_params* p, const double* F, const double stag[3], const double X[3])
{
    long b[3];
    double w[3][ORC_WN];
    for (int a = 0; a < 3; ++a) {
        /* energy-conserving variant (8(f)2): one order lower along the axes this component is staggered on, so that a
         * field that is the discrete gradient of a node potential is gathered as the exact gradient of the order-o
         * interpolation of that potential: d/dx W_o(x - i) = W_{o-1}(x - (i - 1/2)) - W_{o-1}(x - (i + 1/2)) */
        const int order = (p->gather == 1 && stag[a] != 0.0) ? p->order - 1 : p->order;
        b[a] = (long)floor(X[a] - stag[a]) + ORC_WLO;
        for (int t = 0; t < ORC_WN; ++t) w[a][t] = orc_shape(order, X[a] - ((double)(b[a] + t) + stag[a]));
    }
    double acc = 0.0;
    for (int c = 0; c < ORC_WN; ++c) {
        if (w[2][c] == 0.0) continue;
        int k = orc_wrap(b[2] + c, p->nz);
        for (int bb = 0; bb < ORC_WN; ++bb) {
            if (w[1][bb] == 0.0) continue;
            int j = orc_wrap(b[1] + bb, p->ny);
            for (int aa = 0; aa < ORC_WN; ++aa) {
                if (w[0][aa] == 0.0) continue;
                int i = orc_wrap(b[0] + aa, p->nx);
                acc += F[(size_t)i + (size_t)p->nx * ((size_t)j + (size_t)p->ny * (size_t)k)] * w[0][aa] * w[1][bb] * w[2][c];
            }
        }
    }
    return acc;
}

/* Steps 2+3: all six components; fields[c] for c = Ex,Ey,Ez,Bx,By,Bz. out = E then B. */
void orc_gather(const orc_params* p, const double* const fields[6], const double X[3], double out[6])
{
    for (int c = 0; c < 6; ++c) out[c] = orc_gather_component(p, fields[c], ORC_STAG[c], X);
}

/* Step 4: Boris 1970, tan-free t-vector form, h = (q/m) dt/2. */
void orc_boris(const double u[3], const double E[3], const double B[3], double q_over_m, double dt, double u_new[3])
{
    double h = q_over_m * dt * 0.5;
    double um[3], t[3], s[3], up[3], upl[3];
    for (int a = 0; a < 3; ++a) um[a] = u[a] + h * E[a];
    double gm = sqrt(1.0 + um[0] * um[0] + um[1] * um[1] + um[2] * um[2]);
    for (int a = 0; a < 3; ++a) t[a] = h * B[a] / gm;
    double t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
    for (int a = 0; a < 3; ++a) s[a] = 2.0 * t[a] / (1.0 + t2);
    up[0] = um[0] + (um[1] * t[2] - um[2] * t[1]);
    up[1] = um[1] + (um[2] * t[0] - um[0] * t[2]);
    up[2] = um[2] + (um[0] * t[1] - um[1] * t[0]);
    upl[0] = um[0] + (up[1] * s[2] - up[2] * s[1]);
    upl[1] = um[1] + (up[2] * s[0] - up[0] * s[2]);
    upl[2] = um[2] + (up[0] * s[1] - up[1] * s[0]);
    for (int a = 0; a < 3; ++a) u_new[a] = upl[a] + h * E[a];
}

/* Step 5: X' = X + (u/gamma) dt / (dx,dy,dz), unwrapped, in cell units. */
void orc_move(const orc_params* p, const double X[3], const double u[3], double Xn[3])
{
    double g = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    Xn[0] = X[0] + (u[0] / g) * p->dt / p->dx;
    Xn[1] = X[1] + (u[1] / g) * p->dt / p->dy;
    Xn[2] = X[2] + (u[2] / g) * p->dt / p->dz;
}

/* Step 6: Esirkepov 2001 density decomposition for one particle of charge*weight qw
 * moving X0 -> X1 (cell units, |X1-X0| < 1 per axis).  Adds into Jx,Jy,Jz
 * (Jx[i,j,k] sits at (i+1/2,j,k) etc.), node indices wrapped on write. */
void orc_deposit(const orc_params* p, double qw, const double X0[3], const double X1[3],
                 double* Jx, double* Jy, double* Jz)
{
    long b[3];
    double S0[3][ORC_WN], S1[3][ORC_WN], DS[3][ORC_WN];
    for (int a = 0; a < 3; ++a) {
        b[a] = (long)floor(X0[a]) + ORC_WLO;
        for (int t = 0; t < ORC_WN; ++t) {
            double node = (double)(b[a] + t);
            S0[a][t] = orc_shape(p->order, X0[a] - node);
            S1[a][t] = orc_shape(p->order, X1[a] - node);
            DS[a][t] = S1[a][t] - S0[a][t];
        }
    }
    const double V = p->dx * p->dy * p->dz;
    const double cell[3] = {p->dx, p->dy, p->dz};
    double* J[3] = {Jx, Jy, Jz};
    const int n[3] = {p->nx, p->ny, p->nz};
    /* component a flows along axis a; b1,b2 are the other two axes in cyclic order */
    for (int a = 0; a < 3; ++a) {
        const int b1 = (a + 1) % 3, b2 = (a + 2) % 3;
        const double fac = -(qw / V) * (cell[a] / p->dt);
        for (int t2 = 0; t2 < ORC_WN; ++t2) {
            for (int t1 = 0; t1 < ORC_WN; ++t1) {
                double bracket = S0[b1][t1] * S0[b2][t2] + 0.5 * DS[b1][t1] * S0[b2][t2]
                               + 0.5 * S0[b1][t1] * DS[b2][t2] + (1.0 / 3.0) * DS[b1][t1] * DS[b2][t2];
                if (bracket == 0.0) continue;
                double prefix = 0.0;
                /* the last prefix equals sum(DS) = 0 up to round-off and is not written */
                for (int ta = 0; ta < ORC_WN - 1; ++ta) {
                    prefix += DS[a][ta] * bracket;
                    if (prefix == 0.0) continue;
                    long idx[3];
                    idx[a] = b[a] + ta; idx[b1] = b[b1] + t1; idx[b2] = b[b2] + t2;
                    int i = orc_wrap(idx[0], n[0]), j = orc_wrap(idx[1], n[1]), k = orc_wrap(idx[2], n[2]);
                    J[a][(size_t)i + (size_t)n[0] * ((size_t)j + (size_t)n[1] * (size_t)k)] += fac * prefix;
                }
            }
        }
    }
}

/* Charge density at nodes, rho[i,j,k] += qw S(Xx-i) S(Xy-j) S(Xz-k) / V (used by the
 * continuity checks of SURVEY.md §8(c) step 6 pin (i) and reading S22). */
void orc_rho(const orc_params* p, long n, const double* X, const double* Y, const double* Z,
             const double* qw, double* rho)
{
    const double V = p->dx * p->dy * p->dz;
    for (long q = 0; q < n; ++q) {
        double Xp[3] = {X[q], Y[q], Z[q]};
        long b[3];
        double w[3][ORC_WN];
        for (int a = 0; a < 3; ++a) {
            b[a] = (long)floor(Xp[a]) + ORC_WLO;
            for (int t = 0; t < ORC_WN; ++t) w[a][t] = orc_shape(p->order, Xp[a] - (double)(b[a] + t));
        }
        for (int c = 0; c < ORC_WN; ++c) {
            if (w[2][c] == 0.0) continue;
            int k = orc_wrap(b[2] + c, p->nz);
            for (int bb = 0; bb < ORC_WN; ++bb) {
                if (w[1][bb] == 0.0) continue;
                int j = orc_wrap(b[1] + bb, p->ny);
                for (int aa = 0; aa < ORC_WN; ++aa) {
                    if (w[0][aa] == 0.0) continue;
                    int i = orc_wrap(b[0] + aa, p->nx);
                    rho[(size_t)i + (size_t)p->nx * ((size_t)j + (size_t)p->ny * (size_t)k)] += qw[q] / V * w[0][aa] * w[1][bb] * w[2][c];
                }
            }
        }
    }
}

/* Step 7: wrap into [0,N) and compute the supercell index sx + nsx*(sy + nsy*sz). */
int32_t orc_wrap_and_bucket(const orc_params* p, double X[3])
{
    const int n[3] = {p->nx, p->ny, p->nz};
    const int sc[3] = {p->scx, p->scy, p->scz};
    int s[3];
    for (int a = 0; a < 3; ++a) {
        double N = (double)n[a];
        X[a] = X[a] - N * floor(X[a] / N);
        if (X[a] >= N) X[a] = 0.0;          /* rounding of a tiny negative value */
        if (X[a] < 0.0) X[a] = 0.0;
        int cell = (int)floor(X[a]);
        if (cell >= n[a]) cell = n[a] - 1;
        s[a] = cell / sc[a];
    }
    int nsx = p->nx / p->scx, nsy = p->ny / p->scy;
    return s[0] + nsx * (s[1] + nsy * s[2]);
}

/* One full step over n particles (steps 3-7 per particle; particles are independent
 * because E,B are static and J does not feed back).  X,Y,Z are PHYSICAL positions
 * (same units as dx,dy,dz) and are updated in place, as are ux,uy,uz.  J is
 * ACCUMULATED into Jx,Jy,Jz: the caller zeroes it at the start of every step (S16).
 * q[s], m[s] are the species tables.  supercell (may be NULL) receives the new
 * membership.  Returns 0, or -1 if a particle moved >= 1 cell along an axis. */
int orc_step(const orc_params* p, long n,
             double* X, double* Y, double* Z, double* ux, double* uy, double* uz,
             const double* w, const int32_t* species, const double* q, const double* m,
             const double* Ex, const double* Ey, const double* Ez,
             const double* Bx, const double* By, const double* Bz,
             double* Jx, double* Jy, double* Jz, int32_t* supercell)
{
    const double* fields[6] = {Ex, Ey, Ez, Bx, By, Bz};
    int rc = 0;
    for (long i = 0; i < n; ++i) {
        double X0[3] = {X[i] / p->dx, Y[i] / p->dy, Z[i] / p->dz};
        double u[3] = {ux[i], uy[i], uz[i]};
        double F[6], un[3], X1[3];
        int s = species ? species[i] : 0;
        orc_gather(p, fields, X0, F);
        orc_boris(u, F, F + 3, q[s] / m[s], p->dt, un);
        orc_move(p, X0, un, X1);
        for (int a = 0; a < 3; ++a) if (!(fabs(X1[a] - X0[a]) < 1.0)) rc = -1;
        orc_deposit(p, q[s] * w[i], X0, X1, Jx, Jy, Jz);
        int32_t sc = orc_wrap_and_bucket(p, X1);
        X[i] = X1[0] * p->dx; Y[i] = X1[1] * p->dy; Z[i] = X1[2] * p->dz;
        ux[i] = un[0]; uy[i] = un[1]; uz[i] = un[2];
        if (supercell) supercell[i] = sc;
    }
    return rc;
}
