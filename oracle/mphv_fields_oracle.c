/*
 * mphv_fields_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU statement (fp64, no FMA contraction) of what closes the loop around the kinetic hot
 * path of muphyII (arXiv 2305.01487): the FDTD update of Maxwell's equations fed by the species'
 * currents, the interpolation between the staggered field grid and the cell centres the Vlasov
 * sweeps read, and one step of the coupled multi-species Vlasov-Maxwell scheme.
 * Same rules as mphv_oracle.c: only tests/, smoke() and bench.py's CPU legs may call it; it shares no
 * code with the CUDA path.
 *
 * What the paper fixes (PAPER.md, cited "P:Lnnn"):
 *   - eq. (9), P:L91 (sec. 2): curl E = -dB/dt, curl B = mu0 j + mu0 eps0 dE/dt, with the charge
 *     current j = sum_s q_s n_s u_s (and rho = sum_s q_s n_s, div E = rho / eps0).
 *   - P:L141 (sec. 4.1): "Maxwell's equations are solved via the finite difference time domain (FDTD)
 *     method. The two Maxwell's equations that include time derivatives are evolved, and it is, by
 *     construction of the method, ensured that div B = 0."
 *   - P:L147 (sec. 4.2): "The Maxwell solver itself uses Strang splitting between E and B";
 *     "The electron and Maxwell states are integrated using Strang splitting".
 *   - P:L109: a Scheme holds {Vlasov e, Vlasov i, Maxwell}; the models exchange E, B and moments.
 * The paper prints no stencil, no staggering and no boundary rule for the fields; the readings
 * R19..R22 below are listed in DESIGN.md sec. 2.
 *
 * R19 staggering (Yee lattice on the Vlasov cells): integer indices are the CELL CENTRES the Vlasov
 *     model uses (R1, R8). Array element [k][j][i] of
 *         Ex sits at (i+1/2, j, k)      Bx at (i, j+1/2, k+1/2)
 *         Ey sits at (i, j+1/2, k)      By at (i+1/2, j, k+1/2)
 *         Ez sits at (i, j, k+1/2)      Bz at (i+1/2, j+1/2, k)
 *     (E normal to the cell faces, so that div E = rho / eps0 is a difference of face values around a
 *     cell centre where rho lives; B on the cell edges.) An inactive dimension (extent 1) has no
 *     derivative and no staggering along it.
 * R20 interpolation (linear, i.e. arithmetic means of the nearest staggered values):
 *         E_d at a centre   = mean of the 2 face values along d,
 *         B_d at a centre   = mean of the 4 edge values in the plane normal to d,
 *         j_d at an E_d face = mean of the 2 adjacent cell-centre currents.
 * R21 boundary rule of the field arrays: periodic axis = index wrap; bounded ("outflow") axis =
 *     zero-gradient ghost value (the value at the nearest valid index; the rule R6 applies to f).
 * R22 coupled step over dt (leapfrog-like Strang between plasma and Maxwell):
 *         J  = sum_s q_s j_s[f_s]                (moments of the present f_s, R9/R10)
 *         Maxwell(dt/2; J)                       = B(dt/4) E(dt/2; J) B(dt/4)
 *         E_c, B_c = fields at the cell centres (R20)
 *         every species: f_s <- step(dt) with E_c, B_c frozen (mphv_oracle.c, R4/R5)
 *         J' = sum_s q_s j_s[f_s];  Maxwell(dt/2; J').
 *
 * Pins (tests/test_oracle_fields.py): the Yee vacuum dispersion relation sin(w dt/2)/(c dt) =
 * sqrt(sum_d sin^2(k_d dx_d/2)/dx_d^2) (a textbook closed form) through exact return of an eigenmode;
 * div B unchanged to round-off; Gauss's law kept when J obeys the discrete continuity equation;
 * brute-force curl on a 4x3x5 lattice from the definitions of R19 written out with
 * explicit coordinates; interpolation exact for linear fields; Langmuir oscillation at w_p from a
 * cold linear current response; and, through coupled_step (oracle/fields.py) with the Vlasov sweeps, the Landau
 * damping rate and frequency of the k = 0.5 mode (gamma = -0.1533, w = 1.4156: the roots of the
 * plasma dispersion function, computed in the test from scipy.special.wofz), and the dispersion w^2 = w_p^2 + c^2 K^2
 * of a transverse light wave in the same plasma.
 * PARITY UNPINNED against the authors' code: PAPER.md prints no field value of theirs.
 *
 * Layouts: every field array is [3][nz][ny][nx], component-major, C order (as E, B of mphv_oracle.c).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { FLD_BC_PERIODIC = 0, FLD_BC_OUTFLOW = 1 };
enum { FLD_OK = 0, FLD_ERR_ARG = 1 };

typedef struct {
    int32_t nx[3];        /* spatial extents x, y, z; 1 = inactive             */
    int32_t bc[3];        /* per axis: 0 periodic, 1 bounded (zero gradient)   */
    double dx[3];         /* cell widths                                        */
    double c2;            /* c^2 = 1 / (mu0 eps0)                               */
    double inv_eps0;      /* 1 / eps0                                           */
} orc_fgrid;

/* index along one axis after the boundary rule R21 */
static long wrap(long i, int n, int bc)
{
    if (i >= 0 && i < n) return i;
    if (bc == FLD_BC_PERIODIC) { long m = i % n; return m < 0 ? m + n : m; }
    return i < 0 ? 0 : n - 1;
}

/* value of component array a (one of the three [nz][ny][nx] blocks) at (i, j, k) with R21 applied */
static double at(const orc_fgrid *g, const double *a, long i, long j, long k)
{
    const long ii = wrap(i, g->nx[0], g->bc[0]);
    const long jj = wrap(j, g->nx[1], g->bc[1]);
    const long kk = wrap(k, g->nx[2], g->bc[2]);
    return a[(kk * g->nx[1] + jj) * g->nx[0] + ii];
}

/* forward difference (a[idx + 1 along d] - a[idx]) / dx_d; 0 along an inactive axis */
static double dfwd(const orc_fgrid *g, const double *a, int d, long i, long j, long k)
{
    if (g->nx[d] == 1) return 0.0;
    const double hi = at(g, a, i + (d == 0), j + (d == 1), k + (d == 2));
    return (hi - at(g, a, i, j, k)) / g->dx[d];
}
/* backward difference (a[idx] - a[idx - 1 along d]) / dx_d */
static double dbwd(const orc_fgrid *g, const double *a, int d, long i, long j, long k)
{
    if (g->nx[d] == 1) return 0.0;
    const double lo = at(g, a, i - (d == 0), j - (d == 1), k - (d == 2));
    return (at(g, a, i, j, k) - lo) / g->dx[d];
}

static size_t fcount(const orc_fgrid *g) { return (size_t)g->nx[0] * g->nx[1] * g->nx[2]; }

/* Faraday's law, eq. (9): B <- B - dt curl E on the lattice R19. With the positions of R19,
 *   (curl E)_x at (i, j+1/2, k+1/2) = [Ez(i,j+1,k+1/2) - Ez(i,j,k+1/2)]/dy - [Ey(i,j+1/2,k+1) - Ey(i,j+1/2,k)]/dz
 * and cyclic: every difference is a FORWARD difference of the stored arrays. */
int orc_faraday(const orc_fgrid *g, const double *E, double *B, double dt)
{
    if (!g || !E || !B) return FLD_ERR_ARG;
    const size_t ns = fcount(g);
    const double *Ex = E, *Ey = E + ns, *Ez = E + 2 * ns;
    double *Bx = B, *By = B + ns, *Bz = B + 2 * ns;
    for (long k = 0; k < g->nx[2]; ++k)
        for (long j = 0; j < g->nx[1]; ++j)
            for (long i = 0; i < g->nx[0]; ++i) {
                const size_t c = ((size_t)k * g->nx[1] + j) * g->nx[0] + i;
                const double cx = dfwd(g, Ez, 1, i, j, k) - dfwd(g, Ey, 2, i, j, k);
                const double cy = dfwd(g, Ex, 2, i, j, k) - dfwd(g, Ez, 0, i, j, k);
                const double cz = dfwd(g, Ey, 0, i, j, k) - dfwd(g, Ex, 1, i, j, k);
                Bx[c] = Bx[c] - dt * cx;
                By[c] = By[c] - dt * cy;
                Bz[c] = Bz[c] - dt * cz;
            }
    return FLD_OK;
}

/* Ampere-Maxwell law, eq. (9): E <- E + dt (c^2 curl B - J_face / eps0). With R19,
 *   (curl B)_x at (i+1/2, j, k) = [Bz(i+1/2,j+1/2,k) - Bz(i+1/2,j-1/2,k)]/dy - [By(i+1/2,j,k+1/2) - By(i+1/2,j,k-1/2)]/dz
 * and cyclic: every difference is a BACKWARD difference of the stored arrays. J (optional, NULL = vacuum)
 * is the CELL-CENTRED charge current [3][nz][ny][nx]; its value on the face of E_d is the mean of the two
 * adjacent centres along d (R20). */
int orc_ampere(const orc_fgrid *g, double *E, const double *B, const double *J, double dt)
{
    if (!g || !E || !B) return FLD_ERR_ARG;
    const size_t ns = fcount(g);
    double *Ex = E, *Ey = E + ns, *Ez = E + 2 * ns;
    const double *Bx = B, *By = B + ns, *Bz = B + 2 * ns;
    for (long k = 0; k < g->nx[2]; ++k)
        for (long j = 0; j < g->nx[1]; ++j)
            for (long i = 0; i < g->nx[0]; ++i) {
                const size_t c = ((size_t)k * g->nx[1] + j) * g->nx[0] + i;
                const double cx = dbwd(g, Bz, 1, i, j, k) - dbwd(g, By, 2, i, j, k);
                const double cy = dbwd(g, Bx, 2, i, j, k) - dbwd(g, Bz, 0, i, j, k);
                const double cz = dbwd(g, By, 0, i, j, k) - dbwd(g, Bx, 1, i, j, k);
                double jx = 0.0, jy = 0.0, jz = 0.0;
                if (J) {
                    const double *Jx = J, *Jy = J + ns, *Jz = J + 2 * ns;
                    jx = g->nx[0] > 1 ? 0.5 * (Jx[c] + at(g, Jx, i + 1, j, k)) : Jx[c];
                    jy = g->nx[1] > 1 ? 0.5 * (Jy[c] + at(g, Jy, i, j + 1, k)) : Jy[c];
                    jz = g->nx[2] > 1 ? 0.5 * (Jz[c] + at(g, Jz, i, j, k + 1)) : Jz[c];
                }
                Ex[c] = Ex[c] + dt * (g->c2 * cx - g->inv_eps0 * jx);
                Ey[c] = Ey[c] + dt * (g->c2 * cy - g->inv_eps0 * jy);
                Ez[c] = Ez[c] + dt * (g->c2 * cz - g->inv_eps0 * jz);
            }
    return FLD_OK;
}

/* One Maxwell step over dt with the current J frozen: "Strang splitting between E and B":
 * B(dt/2), E(dt; J), B(dt/2). */
int orc_maxwell_step(const orc_fgrid *g, double *E, double *B, const double *J, double dt)
{
    int st;
    if ((st = orc_faraday(g, E, B, 0.5 * dt)) != FLD_OK) return st;
    if ((st = orc_ampere(g, E, B, J, dt)) != FLD_OK) return st;
    return orc_faraday(g, E, B, 0.5 * dt);
}

/* Fields at the cell centres (R20), what mphv_set_fields / orc_step take (R8): Ec, Bc [3][nz][ny][nx]. */
int orc_fields_to_centres(const orc_fgrid *g, const double *E, const double *B, double *Ec, double *Bc)
{
    if (!g || !E || !B || !Ec || !Bc) return FLD_ERR_ARG;
    const size_t ns = fcount(g);
    for (int d = 0; d < 3; ++d) {
        const int a = (d + 1) % 3, b = (d + 2) % 3;       /* the two axes normal to d */
        const double *Ed = E + d * ns, *Bd = B + d * ns;
        for (long k = 0; k < g->nx[2]; ++k)
            for (long j = 0; j < g->nx[1]; ++j)
                for (long i = 0; i < g->nx[0]; ++i) {
                    const size_t c = ((size_t)k * g->nx[1] + j) * g->nx[0] + i;
                    const long id[3] = { i, j, k };
                    /* E_d: faces at id[d] - 1/2 (stored at index id[d] - 1) and id[d] + 1/2 (stored at id[d]) */
                    if (g->nx[d] > 1) {
                        long lo[3] = { i, j, k };
                        lo[d] -= 1;
                        Ec[d * ns + c] = 0.5 * (at(g, Ed, lo[0], lo[1], lo[2]) + Ed[c]);
                    } else {
                        Ec[d * ns + c] = Ed[c];
                    }
                    /* B_d: edges at (id[a] -+ 1/2, id[b] -+ 1/2), stored at offsets -1 / 0 along a and b */
                    double sum = 0.0;
                    int cnt = 0;
                    for (int oa = (g->nx[a] > 1 ? -1 : 0); oa <= 0; ++oa)
                        for (int ob = (g->nx[b] > 1 ? -1 : 0); ob <= 0; ++ob) {
                            long q[3] = { id[0], id[1], id[2] };
                            q[a] += oa; q[b] += ob;
                            sum += at(g, Bd, q[0], q[1], q[2]);
                            ++cnt;
                        }
                    Bc[d * ns + c] = sum / (double)cnt;
                }
    }
    return FLD_OK;
}

/* Charge current of eq. (9): J = sum_s q_s j_s with j_s = int v f_s dv the NUMBER flux of species s (R10).
 * j_all: [nspecies][3][ns] back to back; J: [3][ns]. Summed in species order. */
int orc_charge_current(size_t ns, int nspecies, const double *q, const double *j_all, double *J)
{
    if (!q || !j_all || !J || nspecies < 1) return FLD_ERR_ARG;
    for (size_t e = 0; e < 3 * ns; ++e) {
        double acc = 0.0;
        for (int s = 0; s < nspecies; ++s) acc = acc + q[s] * j_all[(size_t)s * 3 * ns + e];
        J[e] = acc;
    }
    return FLD_OK;
}

/* Discrete divergences on the lattice R19, for the pins and the Gauss-law checks:
 * div E at the cell centres (backward differences of the face values), div B at the cell corners
 * (i+1/2, j+1/2, k+1/2) (forward differences of the edge... face-normal values). out: [nz][ny][nx]. */
int orc_div_E(const orc_fgrid *g, const double *E, double *out)
{
    if (!g || !E || !out) return FLD_ERR_ARG;
    const size_t ns = fcount(g);
    for (long k = 0; k < g->nx[2]; ++k)
        for (long j = 0; j < g->nx[1]; ++j)
            for (long i = 0; i < g->nx[0]; ++i)
                out[((size_t)k * g->nx[1] + j) * g->nx[0] + i] =
                    dbwd(g, E, 0, i, j, k) + dbwd(g, E + ns, 1, i, j, k) + dbwd(g, E + 2 * ns, 2, i, j, k);
    return FLD_OK;
}
int orc_div_B(const orc_fgrid *g, const double *B, double *out)
{
    if (!g || !B || !out) return FLD_ERR_ARG;
    const size_t ns = fcount(g);
    for (long k = 0; k < g->nx[2]; ++k)
        for (long j = 0; j < g->nx[1]; ++j)
            for (long i = 0; i < g->nx[0]; ++i)
                out[((size_t)k * g->nx[1] + j) * g->nx[0] + i] =
                    dfwd(g, B, 0, i, j, k) + dfwd(g, B + ns, 1, i, j, k) + dfwd(g, B + 2 * ns, 2, i, j, k);
    return FLD_OK;
}
