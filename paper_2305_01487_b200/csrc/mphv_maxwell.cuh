// mphv_maxwell.cuh -- the ten-moment Maxwellian (sec. 4.3: "a ten-moment Maxwellian
// distribution, which takes the temperature tensor into account (a multivariate normal distribution)")
// and the exchange of Maxwellians in the two boundary cells of a Vlasov / ten-moment coupling border
// (sigma_1 = 2/3, sigma_2 = 1/3). Readings R16, R17 of DESIGN.md; moment conventions R9, R10:
//   u = j / n,  C_ab = P_ab / n - u_a u_b,
//   M[n,j,P](v) = n (2 pi)^(-D/2) det(C)^(-1/2) exp(-(v-u)^T C^-1 (v-u) / 2)   at the velocity cell centres,
// D = number of active velocity dimensions; n <= 0 or C not positive definite: M = 0.
//   ghost_i = M[fluid data of boundary cell i] + sigma_i (f_ext - M[moments of f_ext]),
// f_ext = the last interior cell of the column (zero-gradient extension).
// One CTA per spatial cell; the 3x3 algebra is done once per CTA by thread 0 and broadcast through
// shared memory, the velocity cube is streamed by all threads along vz pencils (8 bytes written per cell;
// the Gaussian along a pencil by a two-multiplication recurrence with exact restarts, MaxwLine).
#pragma once
#include "mphv_kernels.cuh"

namespace mphv {

struct MaxwCoef { double ux, uy, uz, cxx, cxy, cxz, cyy, cyz, czz, norm; };   // c = -(1/2) C^-1 (off-diagonals doubled)

// Thread-0 setup: coefficients such that M(v) = norm exp(cxx dx^2 + cxy dx dy + ... + czz dz^2), d = v - u.
__device__ inline MaxwCoef maxw_setup(const GridDev &g, double n, double jx, double jy, double jz,
                                      double pxx, double pxy, double pxz, double pyy, double pyz, double pzz)
{
    MaxwCoef m;
    m.ux = m.uy = m.uz = 0.0; m.cxx = m.cxy = m.cxz = m.cyy = m.cyz = m.czz = 0.0; m.norm = 0.0;
    if (!(n > 0.0)) return m;
    const bool ax = g.nv[0] > 1, ay = g.nv[1] > 1, az = g.nv[2] > 1;
    const double in = 1.0 / n;
    const double ux = jx * in, uy = jy * in, uz = jz * in;
    // covariance; an inactive dimension is replaced by a unit variance uncorrelated with the others
    double a = ax ? pxx * in - ux * ux : 1.0, d = ay ? pyy * in - uy * uy : 1.0, f = az ? pzz * in - uz * uz : 1.0;
    double b = (ax && ay) ? pxy * in - ux * uy : 0.0, c = (ax && az) ? pxz * in - ux * uz : 0.0, e = (ay && az) ? pyz * in - uy * uz : 0.0;
    // C = [[a b c], [b d e], [c e f]]: cofactors, determinant, leading minors (Sylvester)
    const double k00 = d * f - e * e, k01 = c * e - b * f, k02 = b * e - c * d;
    const double det = a * k00 + b * k01 + c * k02;
    const double m2 = a * d - b * b;
    if (!(a > 0.0) || !(m2 > 0.0) || !(det > 0.0)) return m;
    const double id = 1.0 / det;
    const double ixx = k00 * id, ixy = k01 * id, ixz = k02 * id;
    const double iyy = (a * f - c * c) * id, iyz = (b * c - a * e) * id, izz = m2 * id;
    const int D = (int)ax + (int)ay + (int)az;
    const double two_pi = 6.283185307179586476925286766559;
    m.norm = n / (pow(two_pi, 0.5 * D) * sqrt(det));
    m.ux = ux; m.uy = uy; m.uz = uz;
    m.cxx = ax ? -0.5 * ixx : 0.0; m.cyy = ay ? -0.5 * iyy : 0.0; m.czz = az ? -0.5 * izz : 0.0;
    m.cxy = (ax && ay) ? -ixy : 0.0; m.cxz = (ax && az) ? -ixz : 0.0; m.cyz = (ay && az) ? -iyz : 0.0;
    return m;
}

__device__ __forceinline__ double maxw_eval(const MaxwCoef &m, double vx, double vy, double vz)
{
    const double dx = vx - m.ux, dy = vy - m.uy, dz = vz - m.uz;
    const double q = dx * (m.cxx * dx + m.cxy * dy + m.cxz * dz) + dy * (m.cyy * dy + m.cyz * dz) + m.czz * dz * dz;
    return m.norm * exp(q);
}

// A Maxwellian along one vz pencil (vx, vy fixed): q(vz) is quadratic in vz, so consecutive cells follow from
// two multiplications, e_{k+1} = e_k r_k, r_{k+1} = r_k rho with rho = exp(2 czz dvz^2); e and r are re-evaluated
// exactly every MAXW_RS cells, which bounds the accumulated rounding to ~(RS^2/2) ulp (4e-15) and keeps
// underflow local. One exp per cell becomes 2/RS.
enum { MAXW_RS = 8 };
struct MaxwLine {
    double a0, b, e, r, rho;
    double czz, norm, uz;            // for the direct evaluation of a block the recurrence cannot carry
    bool direct;
    __device__ __forceinline__ void init(const MaxwCoef &m, double vx, double vy, double dvz_)
    {
        const double dx = vx - m.ux, dy = vy - m.uy;
        a0 = dx * (m.cxx * dx + m.cxy * dy) + m.cyy * dy * dy;
        b = m.cxz * dx + m.cyz * dy;
        rho = exp(2.0 * m.czz * dvz_ * dvz_);
        e = 0.0; r = 0.0;
        czz = m.czz; norm = m.norm; uz = m.uz; direct = false;
    }
    __device__ __forceinline__ void restart(const MaxwCoef &m, double vz, double dvz_)
    {
        const double dz = vz - m.uz;
        e = m.norm * exp(a0 + dz * (b + m.czz * dz));
        r = exp(dvz_ * (b + m.czz * (2.0 * dz + dvz_)));
        // A cold or unresolved Maxwellian (thermal spread << dvz): e underflows while r overflows and the
        // recurrence would write 0 * inf = NaN, or lose the cells that come back above the underflow threshold
        // inside the block. Such blocks are evaluated cell by cell (one exp each), like the definition.
        direct = !(e > 1e-250 && r > 1e-25 && r < 1e25);
    }
    // the value at the next cell of the pencil by the recurrence (only while !direct)
    __device__ __forceinline__ double next() { const double v = e; e *= r; r *= rho; return v; }
    // the value at cell jz by the definition (one exp): what a block with `direct` set must use
    __device__ __forceinline__ double eval(const GridDev &g, int jz) const
    {
        const double dz = vcentre(g, 2, jz) - uz;
        return norm * exp(a0 + dz * (b + czz * dz));
    }
};

struct MaxwArgs {
    const double *n, *j, *P;    // [count], [3][count], [6][count]
    long long count;
    double *f_out;              // [count][nvel]
    GridDev g;
};

__global__ void __launch_bounds__(512)
maxwellian_kernel(const MaxwArgs p)
{
    __shared__ MaxwCoef sm;
    const GridDev &g = p.g;
    const long long c = blockIdx.x, cnt = p.count;
    if (threadIdx.x == 0)
        sm = maxw_setup(g, p.n[c], p.j[c], p.j[cnt + c], p.j[2 * cnt + c],
                        p.P[c], p.P[cnt + c], p.P[2 * cnt + c], p.P[3 * cnt + c], p.P[4 * cnt + c], p.P[5 * cnt + c]);
    __syncthreads();
    const MaxwCoef m = sm;
    double *cube = p.f_out + c * g.nvel;
    const int plane = g.nv[0] * g.nv[1];
    for (int pos = threadIdx.x; pos < plane; pos += blockDim.x) {
        const int jy = pos / g.nv[0], jx = pos - jy * g.nv[0];
        const double vx = vcentre(g, 0, jx), vy = vcentre(g, 1, jy);
        MaxwLine ln;
        ln.init(m, vx, vy, g.dv[2]);
        for (int j0 = 0; j0 < g.nv[2]; j0 += MAXW_RS) {
            ln.restart(m, vcentre(g, 2, j0), g.dv[2]);
            if (ln.direct && m.norm > 0.0) {               // a cold Maxwellian: this block by the definition
                for (int u = 0; u < MAXW_RS && j0 + u < g.nv[2]; ++u) cube[(long long)(j0 + u) * plane + pos] = ln.eval(g, j0 + u);
                continue;
            }
#pragma unroll
            for (int u = 0; u < MAXW_RS; ++u) {
                const double v = m.norm > 0.0 ? ln.next() : 0.0;
                if (j0 + u < g.nv[2]) cube[(long long)(j0 + u) * plane + pos] = v;
            }
        }
    }
}

struct ExchArgs {
    double *f;                  // the block, in place
    const double *n_fl, *j_fl, *P_fl;   // [2][plane], [3][2][plane], [6][2][plane]
    long long plane;            // spatial cells per layer
    long long sa, sb, sd;       // strides (in spatial cells) of the two plane indices and of the swept dim
    int na;                     // extent of the faster plane index
    int n;                      // extent along dim
    int side;
    GridDev g;
};

// grid = 2 plane CTAs: blockIdx.x = layer * plane + pl
__global__ void __launch_bounds__(512)
exchange_kernel(const ExchArgs p)
{
    __shared__ double red[10 * 32];
    __shared__ MaxwCoef sm[2];
    const GridDev &g = p.g;
    const int layer = (int)(blockIdx.x / p.plane);
    const long long pl = blockIdx.x - (long long)layer * p.plane;
    const long long ib = pl / p.na, ia = pl - ib * p.na;
    const long long col = ia * p.sa + ib * p.sb;
    const int interior = p.side ? p.n - 3 : 2;
    const int idx = p.side ? p.n - 2 + layer : layer;
    const int dist = p.side ? layer + 1 : 2 - layer;                     // 1 = next to the interior
    const double sigma = dist == 1 ? 2.0 / 3.0 : 1.0 / 3.0;
    const double *fext = p.f + (col + interior * p.sd) * g.nvel;
    double *dst = p.f + (col + idx * p.sd) * g.nvel;
    const int plane = g.nv[0] * g.nv[1];

    // moments of f_ext (midpoint rule, separable accumulation along vz)
    double m[10];
#pragma unroll
    for (int k = 0; k < 10; ++k) m[k] = 0.0;
    for (int pos = threadIdx.x; pos < plane; pos += blockDim.x) {
        const int jy = pos / g.nv[0], jx = pos - jy * g.nv[0];
        const double vx = vcentre(g, 0, jx), vy = vcentre(g, 1, jy);
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;
        for (int j0 = 0; j0 < g.nv[2]; j0 += 8) {
            double fv[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) fv[u] = j0 + u < g.nv[2] ? fext[(long long)(j0 + u) * plane + pos] : 0.0;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const double vz = vcentre(g, 2, j0 + u);
                const double t = vz * fv[u];
                s0 += fv[u]; s1 += t; s2 = fma(vz, t, s2);
            }
        }
        const double x0 = vx * s0, y0 = vy * s0;
        m[0] += s0;
        m[1] += x0; m[2] += y0; m[3] += s1;
        m[4] = fma(vx, x0, m[4]); m[5] = fma(vx, y0, m[5]); m[6] = fma(vx, s1, m[6]);
        m[7] = fma(vy, y0, m[7]); m[8] = fma(vy, s1, m[8]); m[9] += s2;
    }
    block_reduce_sum<10>(m, red);
    if (threadIdx.x == 0) {
        const double dV = g.dv[0] * g.dv[1] * g.dv[2];
        sm[0] = maxw_setup(g, m[0] * dV, m[1] * dV, m[2] * dV, m[3] * dV, m[4] * dV, m[5] * dV, m[6] * dV,
                           m[7] * dV, m[8] * dV, m[9] * dV);
        const long long k = (long long)layer * p.plane + pl, L = 2 * p.plane;
        sm[1] = maxw_setup(g, p.n_fl[k], p.j_fl[k], p.j_fl[L + k], p.j_fl[2 * L + k],
                           p.P_fl[k], p.P_fl[L + k], p.P_fl[2 * L + k], p.P_fl[3 * L + k], p.P_fl[4 * L + k], p.P_fl[5 * L + k]);
    }
    __syncthreads();
    const MaxwCoef mex = sm[0], mfl = sm[1];
    for (int pos = threadIdx.x; pos < plane; pos += blockDim.x) {
        const int jy = pos / g.nv[0], jx = pos - jy * g.nv[0];
        const double vx = vcentre(g, 0, jx), vy = vcentre(g, 1, jy);
        MaxwLine la, lb;
        la.init(mfl, vx, vy, g.dv[2]); lb.init(mex, vx, vy, g.dv[2]);
        for (int j0 = 0; j0 < g.nv[2]; j0 += MAXW_RS) {
            const double vz = vcentre(g, 2, j0);
            la.restart(mfl, vz, g.dv[2]); lb.restart(mex, vz, g.dv[2]);
            double fv[MAXW_RS];
#pragma unroll
            for (int u = 0; u < MAXW_RS; ++u) fv[u] = j0 + u < g.nv[2] ? fext[(long long)(j0 + u) * plane + pos] : 0.0;
            if (la.direct || lb.direct) {                  // a cold Maxwellian: this block by the definition
                for (int u = 0; u < MAXW_RS && j0 + u < g.nv[2]; ++u) {
                    const double a = mfl.norm > 0.0 ? la.eval(g, j0 + u) : 0.0;
                    const double b = mex.norm > 0.0 ? lb.eval(g, j0 + u) : 0.0;
                    dst[(long long)(j0 + u) * plane + pos] = a + sigma * (fv[u] - b);
                }
                continue;
            }
#pragma unroll
            for (int u = 0; u < MAXW_RS; ++u) {
                const double a = mfl.norm > 0.0 ? la.next() : 0.0;
                const double b = mex.norm > 0.0 ? lb.next() : 0.0;
                if (j0 + u < g.nv[2]) dst[(long long)(j0 + u) * plane + pos] = a + sigma * (fv[u] - b);
            }
        }
    }
}

// ---------------------------------------------------------------- moment matching (R18)
// f <- M[n_t, j_t, P_t] + (f - M[moments of f]) in every spatial cell, in place: one CTA per cell, the
// cube is read twice (moments, then the update; the second read comes from L2 for the cubes still resident).
struct MatchArgs {
    double *f;
    const double *n_t, *j_t, *P_t;      // [ns], [3][ns], [6][ns]
    GridDev g;
};

__global__ void __launch_bounds__(512)
match_kernel(const MatchArgs p)
{
    __shared__ double red[10 * 32];
    __shared__ MaxwCoef sm[2];
    const GridDev &g = p.g;
    const long long cell = blockIdx.x, ns = g.ns;
    double *cube = p.f + cell * g.nvel;
    const int plane = g.nv[0] * g.nv[1];
    double m[10];
#pragma unroll
    for (int k = 0; k < 10; ++k) m[k] = 0.0;
    for (int pos = threadIdx.x; pos < plane; pos += blockDim.x) {
        const int jy = pos / g.nv[0], jx = pos - jy * g.nv[0];
        const double vx = vcentre(g, 0, jx), vy = vcentre(g, 1, jy);
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;
        for (int j0 = 0; j0 < g.nv[2]; j0 += 8) {
            double fv[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) fv[u] = j0 + u < g.nv[2] ? cube[(long long)(j0 + u) * plane + pos] : 0.0;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const double vz = vcentre(g, 2, j0 + u);
                const double t = vz * fv[u];
                s0 += fv[u]; s1 += t; s2 = fma(vz, t, s2);
            }
        }
        const double x0 = vx * s0, y0 = vy * s0;
        m[0] += s0;
        m[1] += x0; m[2] += y0; m[3] += s1;
        m[4] = fma(vx, x0, m[4]); m[5] = fma(vx, y0, m[5]); m[6] = fma(vx, s1, m[6]);
        m[7] = fma(vy, y0, m[7]); m[8] = fma(vy, s1, m[8]); m[9] += s2;
    }
    block_reduce_sum<10>(m, red);
    if (threadIdx.x == 0) {
        const double dV = g.dv[0] * g.dv[1] * g.dv[2];
        sm[0] = maxw_setup(g, m[0] * dV, m[1] * dV, m[2] * dV, m[3] * dV, m[4] * dV, m[5] * dV, m[6] * dV,
                           m[7] * dV, m[8] * dV, m[9] * dV);
        sm[1] = maxw_setup(g, p.n_t[cell], p.j_t[cell], p.j_t[ns + cell], p.j_t[2 * ns + cell],
                           p.P_t[cell], p.P_t[ns + cell], p.P_t[2 * ns + cell], p.P_t[3 * ns + cell],
                           p.P_t[4 * ns + cell], p.P_t[5 * ns + cell]);
    }
    __syncthreads();
    const MaxwCoef mf = sm[0], mt = sm[1];
    for (int pos = threadIdx.x; pos < plane; pos += blockDim.x) {
        const int jy = pos / g.nv[0], jx = pos - jy * g.nv[0];
        const double vx = vcentre(g, 0, jx), vy = vcentre(g, 1, jy);
        MaxwLine la, lb;
        la.init(mt, vx, vy, g.dv[2]); lb.init(mf, vx, vy, g.dv[2]);
        for (int j0 = 0; j0 < g.nv[2]; j0 += MAXW_RS) {
            const double vz = vcentre(g, 2, j0);
            la.restart(mt, vz, g.dv[2]); lb.restart(mf, vz, g.dv[2]);
            double fv[MAXW_RS];
#pragma unroll
            for (int u = 0; u < MAXW_RS; ++u) fv[u] = j0 + u < g.nv[2] ? cube[(long long)(j0 + u) * plane + pos] : 0.0;
            if (la.direct || lb.direct) {                  // a cold Maxwellian: this block by the definition
                for (int u = 0; u < MAXW_RS && j0 + u < g.nv[2]; ++u) {
                    const double a = mt.norm > 0.0 ? la.eval(g, j0 + u) : 0.0;
                    const double b = mf.norm > 0.0 ? lb.eval(g, j0 + u) : 0.0;
                    cube[(long long)(j0 + u) * plane + pos] = a + (fv[u] - b);
                }
                continue;
            }
#pragma unroll
            for (int u = 0; u < MAXW_RS; ++u) {
                const double a = mt.norm > 0.0 ? la.next() : 0.0;
                const double b = mf.norm > 0.0 ? lb.next() : 0.0;
                if (j0 + u < g.nv[2]) cube[(long long)(j0 + u) * plane + pos] = a + (fv[u] - b);
            }
        }
    }
}

}  // namespace mphv
