// mphv_fields.cuh -- the field side of a coupled run: FDTD update of Maxwell's equations
// (eq. (9); "solved via the finite difference time domain (FDTD) method"; "Strang splitting between
// E and B"), interpolation of the staggered fields to the cell centres the Vlasov sweeps read, and the charge
// current J = sum_s q_s j_s. Readings R19 (Yee lattice on the Vlasov cells: E_d on the faces normal to d, B_d on
// the edges along d), R20 (arithmetic means between the lattices), R21 (periodic wrap / zero-gradient ghost) of
// DESIGN.md. O(spatial cells) work: these kernels are latency-bound, so the whole Maxwell(dt) update with its
// current and the centring runs as ONE single-CTA launch when the grid is small enough (maxwell_fused_kernel),
// else as one launch per phase. Shares no code with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mphv {

enum { FLD_MAX_SPECIES = 4 };

struct FieldDev {
    int nx[3], bc[3];               // bc: 0 periodic, 1 zero gradient (R21)
    double inv_dx[3];               // 1 / dx_d, 0 along an inactive axis (no derivative there)
    double c2, inv_eps0;
    long long ns;
};

struct MaxwellArgs {
    FieldDev g;
    double *E, *B;                  // staggered, [3][ns]
    const double *J;                // cell-centred charge current [3][ns] or NULL (vacuum)
    double *Jout;                   // fused kernel: where sum_s q_s j_s is written (NULL: use J as given)
    int nspecies;
    double q[FLD_MAX_SPECIES];
    const double *j[FLD_MAX_SPECIES];   // number fluxes of the species, [3][ns] each
    double dt;                      // Maxwell step: B(dt/2) E(dt) B(dt/2)
    int reps;                       // fused kernel: that many Maxwell steps back to back with the same J
    double *Ec, *Bc;                // centred output [3][ns] (NULL: skip)
};

__device__ __forceinline__ int fld_wrap(int i, int n, int bc)
{
    if (i >= 0 && i < n) return i;
    if (bc == 0) return i < 0 ? i + n : i - n;      // neighbours only: |i - valid| <= 1
    return i < 0 ? 0 : n - 1;
}

struct CellIdx { int i, j, k; long long c; };

__device__ __forceinline__ CellIdx fld_cell(const FieldDev &g, long long c)
{
    CellIdx x;
    x.c = c;
    x.i = (int)(c % g.nx[0]);
    const long long r = c / g.nx[0];
    x.j = (int)(r % g.nx[1]);
    x.k = (int)(r / g.nx[1]);
    return x;
}

// linear index of the neighbour displaced by o (= -1, 0, +1) along axis d, boundary rule applied
__device__ __forceinline__ long long fld_nb(const FieldDev &g, const CellIdx &x, int d, int o)
{
    const int i = d == 0 ? fld_wrap(x.i + o, g.nx[0], g.bc[0]) : x.i;
    const int j = d == 1 ? fld_wrap(x.j + o, g.nx[1], g.bc[1]) : x.j;
    const int k = d == 2 ? fld_wrap(x.k + o, g.nx[2], g.bc[2]) : x.k;
    return ((long long)k * g.nx[1] + j) * g.nx[0] + i;
}

// forward / backward difference quotient of component array a along axis d at cell x
__device__ __forceinline__ double fld_dfwd(const FieldDev &g, const double *a, const CellIdx &x, int d)
{
    if (g.nx[d] == 1) return 0.0;
    return __dmul_rn(__dsub_rn(a[fld_nb(g, x, d, +1)], a[x.c]), g.inv_dx[d]);
}
__device__ __forceinline__ double fld_dbwd(const FieldDev &g, const double *a, const CellIdx &x, int d)
{
    if (g.nx[d] == 1) return 0.0;
    return __dmul_rn(__dsub_rn(a[x.c], a[fld_nb(g, x, d, -1)]), g.inv_dx[d]);
}

// Faraday: B <- B - dt curl E; every difference is a forward difference of the stored arrays (R19)
__device__ __forceinline__ void faraday_cell(const FieldDev &g, const double *E, double *B, double dt, long long c)
{
    const CellIdx x = fld_cell(g, c);
    const double *Ex = E, *Ey = E + g.ns, *Ez = E + 2 * g.ns;
    const double cx = fld_dfwd(g, Ez, x, 1) - fld_dfwd(g, Ey, x, 2);
    const double cy = fld_dfwd(g, Ex, x, 2) - fld_dfwd(g, Ez, x, 0);
    const double cz = fld_dfwd(g, Ey, x, 0) - fld_dfwd(g, Ex, x, 1);
    B[c] = fma(-dt, cx, B[c]);
    B[g.ns + c] = fma(-dt, cy, B[g.ns + c]);
    B[2 * g.ns + c] = fma(-dt, cz, B[2 * g.ns + c]);
}

// Ampere-Maxwell: E <- E + dt (c^2 curl B - J_face / eps0); backward differences; J_face = mean of the two cells
__device__ __forceinline__ void ampere_cell(const FieldDev &g, double *E, const double *B, const double *J, double dt, long long c)
{
    const CellIdx x = fld_cell(g, c);
    const double *Bx = B, *By = B + g.ns, *Bz = B + 2 * g.ns;
    const double cx = fld_dbwd(g, Bz, x, 1) - fld_dbwd(g, By, x, 2);
    const double cy = fld_dbwd(g, Bx, x, 2) - fld_dbwd(g, Bz, x, 0);
    const double cz = fld_dbwd(g, By, x, 0) - fld_dbwd(g, Bx, x, 1);
    double jf[3] = { 0.0, 0.0, 0.0 };
    if (J) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double *Jd = J + d * g.ns;
            jf[d] = g.nx[d] > 1 ? 0.5 * (Jd[c] + Jd[fld_nb(g, x, d, +1)]) : Jd[c];
        }
    }
    E[c] = fma(dt, g.c2 * cx - g.inv_eps0 * jf[0], E[c]);
    E[g.ns + c] = fma(dt, g.c2 * cy - g.inv_eps0 * jf[1], E[g.ns + c]);
    E[2 * g.ns + c] = fma(dt, g.c2 * cz - g.inv_eps0 * jf[2], E[2 * g.ns + c]);
}

// centred fields (R20): E_d = mean of its two faces along d, B_d = mean of its four edges in the plane normal to d
__device__ __forceinline__ void centre_cell(const FieldDev &g, const double *E, const double *B, double *Ec, double *Bc, long long c)
{
    const CellIdx x = fld_cell(g, c);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int a = (d + 1) % 3, b = (d + 2) % 3;
        const double *Ed = E + d * g.ns, *Bd = B + d * g.ns;
        Ec[d * g.ns + c] = g.nx[d] > 1 ? 0.5 * (Ed[fld_nb(g, x, d, -1)] + Ed[c]) : Ed[c];
        const bool aa = g.nx[a] > 1, ab = g.nx[b] > 1;
        double v;
        if (aa && ab) {
            const CellIdx xa = fld_cell(g, fld_nb(g, x, a, -1));
            v = 0.25 * ((Bd[fld_nb(g, xa, b, -1)] + Bd[xa.c]) + (Bd[fld_nb(g, x, b, -1)] + Bd[c]));
        } else if (aa) {
            v = 0.5 * (Bd[fld_nb(g, x, a, -1)] + Bd[c]);
        } else if (ab) {
            v = 0.5 * (Bd[fld_nb(g, x, b, -1)] + Bd[c]);
        } else {
            v = Bd[c];
        }
        Bc[d * g.ns + c] = v;
    }
}

__device__ __forceinline__ void current_entry(const MaxwellArgs &p, long long e)
{
    double acc = 0.0;
    for (int s = 0; s < p.nspecies; ++s) acc = fma(p.q[s], p.j[s][e], acc);
    p.Jout[e] = acc;
}

// ---- one launch per phase (any grid size)
__global__ void __launch_bounds__(256) faraday_kernel(MaxwellArgs p, double dt)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < p.g.ns) faraday_cell(p.g, p.E, p.B, dt, c);
}
__global__ void __launch_bounds__(256) ampere_kernel(MaxwellArgs p, double dt)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < p.g.ns) ampere_cell(p.g, p.E, p.B, p.J, dt, c);
}
__global__ void __launch_bounds__(256) centre_kernel(MaxwellArgs p)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < p.g.ns) centre_cell(p.g, p.E, p.B, p.Ec, p.Bc, c);
}
__global__ void __launch_bounds__(256) current_kernel(MaxwellArgs p)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < 3 * p.g.ns) current_entry(p, e);
}

// ---- everything in one single-CTA launch: [J = sum q_s j_s], reps x [B(dt/2) E(dt; J) B(dt/2)], [centring].
// The phases depend on neighbouring cells, so they are separated by __syncthreads (one CTA: global writes of a
// phase are visible to the whole block after the barrier). Two Faraday half steps that meet are NOT merged, so
// the result is bitwise that of the per-phase launches.
__global__ void __launch_bounds__(1024) maxwell_fused_kernel(MaxwellArgs p)
{
    const long long ns = p.g.ns;
    const double *J = p.J;
    if (p.Jout) {
        for (long long e = threadIdx.x; e < 3 * ns; e += blockDim.x) current_entry(p, e);
        J = p.Jout;
        __syncthreads();
    }
    for (int r = 0; r < p.reps; ++r) {
        for (long long c = threadIdx.x; c < ns; c += blockDim.x) faraday_cell(p.g, p.E, p.B, 0.5 * p.dt, c);
        __syncthreads();
        for (long long c = threadIdx.x; c < ns; c += blockDim.x) ampere_cell(p.g, p.E, p.B, J, p.dt, c);
        __syncthreads();
        for (long long c = threadIdx.x; c < ns; c += blockDim.x) faraday_cell(p.g, p.E, p.B, 0.5 * p.dt, c);
        __syncthreads();
    }
    if (p.Ec)
        for (long long c = threadIdx.x; c < ns; c += blockDim.x) centre_cell(p.g, p.E, p.B, p.Ec, p.Bc, c);
}

}  // namespace mphv
