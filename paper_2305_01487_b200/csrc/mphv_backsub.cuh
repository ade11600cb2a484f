// mphv_backsub.cuh -- the V stage "realized via backsubstitution" (sec. 4.1), reading R15
// of DESIGN.md: three 1-D conservative remaps along vx, vy, vz whose composition is the exact
// characteristic foot of dv/dt = (q/m)(E + v x B) over dt (Boris rotation, fields frozen), instead of
// the three plain shifts a_d dt of the default mode.
//
// With v = R V + c the Boris map of a spatial cell (R = I + S + S T, (T u) = u x t, (S u) = u x s,
// t = (q/m)(dt/2) B, s = 2 t / (1 + t^2), c = (I + R)(q/m)(dt/2) E), sweep d displaces the face at
// coordinate xi of a pencil by an AFFINE function of xi and of the pencil's two other coordinates:
//     s_face = (xi - foot_d) / dv_d = K0 + K1 xi + Ka va + Kb vb,
//     d = vx: foot = (xi - c_x - R_xy vy - R_xz vz) / R_xx                       (va, vb) = (vy, vz)
//     d = vy: foot = (xi - c_y - R_yx (vx - c_x - R_xz vz)/R_xx - R_yz vz) / D,   D = R_yy - R_yx R_xy / R_xx
//                                                                                 (va, vb) = (vx, vz)
//     d = vz: foot = R_xz (vx - c_x) + R_yz (vy - c_y) + R_zz (xi - c_z)         (va, vb) = (vx, vy)
// backsub_coeff_kernel evaluates the 12 numbers K per spatial cell once per (fields, dt); the differences
// 1 - 1/R_xx, 1 - 1/D, 1 - R_zz are formed from R - I = S + S T, never by subtracting from 1.
// The sweep kernels are face-form PFC-3 remaps (R2, R3, R7) with one Courant number per face:
//   bs_march_kernel   strided axes vy, vz: one thread per VEC adjacent pencils, register window,
//                     loads U steps ahead;
//   bs_vx_kernel      contiguous axis vx: one thread per CH cells of a row, all loads -> barrier -> stores.
#pragma once
#include "mphv_kernels.cuh"

namespace mphv {

struct BacksubArgs {
    double *f;
    const double *K;        // [ns][12]: sweep d at K + 12 cell + 4 d: K0, K1, Ka, Kb
    GridDev g;
};

// ---------------------------------------------------------------- coefficients and range check
// smax[d] (bit pattern of a non-negative double, atomicMax) = max |s_face| over the interior faces of
// sweep d; the extreme of an affine function over the box of (xi, va, vb) is at a corner.
__global__ void __launch_bounds__(128)
backsub_coeff_kernel(const double *__restrict__ E, const double *__restrict__ B, GridDev g, double dt,
                     double *__restrict__ K, unsigned long long *__restrict__ smax)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double mx[3] = { 0.0, 0.0, 0.0 };
    if (cell < g.ns) {
        const double h = 0.5 * g.qm * dt;
        const double tx = h * B[cell], ty = h * B[g.ns + cell], tz = h * B[2 * g.ns + cell];
        const double w = 2.0 / (1.0 + (tx * tx + ty * ty + tz * tz));
        const double sx = w * tx, sy = w * ty, sz = w * tz;
        // A = R - I = S + S T, with S = [[0, sz, -sy], [-sz, 0, sx], [sy, -sx, 0]] (same shape for T)
        const double Axx = -(sz * tz + sy * ty), Axy = sz + sy * tx, Axz = -sy + sz * tx;
        const double Ayx = -sz + sx * ty, Ayy = -(sz * tz + sx * tx), Ayz = sx + sz * ty;
        const double Azx = sy + sx * tz, Azy = -sx + sy * tz, Azz = -(sy * ty + sx * tx);
        const double Rxx = 1.0 + Axx;
        const double hx = h * E[cell], hy = h * E[g.ns + cell], hz = h * E[2 * g.ns + cell];
        // c = (I + R) hE = 2 hE + A hE
        const double cx = 2.0 * hx + (Axx * hx + Axy * hy + Axz * hz);
        const double cy = 2.0 * hy + (Ayx * hx + Ayy * hy + Ayz * hz);
        const double cz = 2.0 * hz + (Azx * hx + Azy * hy + Azz * hz);
        double k[12];
        // vx: delta = xi Axx / Rxx + (cx + Axy vy + Axz vz) / Rxx
        const double ix = 1.0 / (Rxx * g.dv[0]);
        k[0] = cx * ix; k[1] = Axx * ix; k[2] = Axy * ix; k[3] = Axz * ix;
        // vy: D - 1 = Ayy - Ayx Axy / Rxx;  delta = xi (D - 1)/D + [cy + Ayx (vx - cx - Axz vz)/Rxx + Ayz vz] / D
        const double r = Ayx / Rxx;
        const double Dm1 = Ayy - r * Axy;
        const double iy = 1.0 / ((1.0 + Dm1) * g.dv[1]);
        k[4] = (cy - r * cx) * iy; k[5] = Dm1 * iy; k[6] = r * iy; k[7] = (Ayz - r * Axz) * iy;
        // vz: delta = -xi Azz - Axz (vx - cx) - Ayz (vy - cy) + (1 + Azz) cz
        const double iz = 1.0 / g.dv[2];
        k[8] = (Axz * cx + Ayz * cy + (1.0 + Azz) * cz) * iz; k[9] = -Azz * iz; k[10] = -Axz * iz; k[11] = -Ayz * iz;
#pragma unroll
        for (int i = 0; i < 12; ++i) K[cell * 12 + i] = k[i];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int da = d == 0 ? 1 : 0, db = d == 2 ? 1 : 2;
            for (int corner = 0; corner < 8; ++corner) {
                const double xi = g.vlo[d] + (corner & 1 ? (double)(g.nv[d] - 1) : 1.0) * g.dv[d];   // interior faces
                const double va = vcentre(g, da, corner & 2 ? g.nv[da] - 1 : 0);
                const double vb = vcentre(g, db, corner & 4 ? g.nv[db] - 1 : 0);
                const double s = fabs(k[4 * d] + k[4 * d + 1] * xi + k[4 * d + 2] * va + k[4 * d + 3] * vb);
                mx[d] = (s == s) ? fmax(mx[d], s) : __longlong_as_double(0x7ff0000000000000LL);
            }
        }
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double x = mx[d];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x = fmax(x, __shfl_down_sync(0xffffffffu, x, off));
        if ((threadIdx.x & 31) == 0) atomicMax(smax + d, (unsigned long long)__double_as_longlong(x));
    }
}

// Flux through one face with its own Courant number s (|s| < 1): upwind triple by the sign of s.
// w0..w3 = g_{i-1}, g_i, g_{i+1}, g_{i+2} around face i+1/2.
__device__ __forceinline__ double bs_face_flux(double w0, double w1, double w2, double w3, double s)
{
    const double fr = fabs(s), om = 1.0 - fr;
    const double c1 = (om * (2.0 - fr)) * (1.0 / 6.0);
    const double c2 = (om * (1.0 + fr)) * (1.0 / 6.0);
    const bool ps = __double2hiint(s) >= 0;
    return face_flux(ps ? w0 : w3, ps ? w1 : w2, ps ? w2 : w1, s, c1, c2);
}

// VEC faces of one march step. The face displacement is affine along the pencil, so the sign of s rarely
// changes inside a warp: where every lane agrees the upwind triple needs no selects.
template <int VEC>
__device__ __forceinline__ void bs_face_fluxes(const double *w0, const double *w1, const double *w2, const double *w3,
                                               const double *s, double *ph)
{
    bool allpos = true, allneg = true;
#pragma unroll
    for (int l = 0; l < VEC; ++l) { const bool ps = __double2hiint(s[l]) >= 0; allpos = allpos && ps; allneg = allneg && !ps; }
    const unsigned mask = __activemask();
    if (__all_sync(mask, allpos)) {
#pragma unroll
        for (int l = 0; l < VEC; ++l) {
            const double fr = fabs(s[l]), om = 1.0 - fr;
            ph[l] = face_flux(w0[l], w1[l], w2[l], s[l], (om * (2.0 - fr)) * (1.0 / 6.0), (om * (1.0 + fr)) * (1.0 / 6.0));
        }
    } else if (__all_sync(mask, allneg)) {
#pragma unroll
        for (int l = 0; l < VEC; ++l) {
            const double fr = fabs(s[l]), om = 1.0 - fr;
            ph[l] = face_flux(w3[l], w2[l], w1[l], s[l], (om * (2.0 - fr)) * (1.0 / 6.0), (om * (1.0 + fr)) * (1.0 / 6.0));
        }
    } else {
#pragma unroll
        for (int l = 0; l < VEC; ++l) ph[l] = bs_face_flux(w0[l], w1[l], w2[l], w3[l], s[l]);
    }
}

// ---------------------------------------------------------------- strided axes vy, vz
// f viewed as [outer][n][inner]: dim 1: outer = (cell, jz), inner = nvx; dim 2: outer = cell, inner = nvy nvx.
template <int VEC, int U>
__global__ void __launch_bounds__(256)
bs_march_kernel(const BacksubArgs p, int dim, long long outer, int n, long long inner)
{
    typedef V<VEC> T;
    const long long innerV = inner / VEC;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= outer * innerV) return;
    const long long o = t / innerV;
    const long long e0 = (t - o * innerV) * VEC;
    const GridDev &g = p.g;
    double *base = p.f + (o * n) * inner + e0;

    // Courant number of face i+1/2: sA + (i + 1) sB
    double sA[VEC], sB;
    {
        long long cell; double va[VEC], vb[VEC];
        if (dim == 2) {
            cell = o;
#pragma unroll
            for (int l = 0; l < VEC; ++l) {
                const long long e = e0 + l;
                const int jy = (int)(e / g.nv[0]), jx = (int)(e - (long long)jy * g.nv[0]);
                va[l] = vcentre(g, 0, jx); vb[l] = vcentre(g, 1, jy);
            }
        } else {
            cell = o / g.nv[2];
            const int jz = (int)(o - cell * g.nv[2]);
#pragma unroll
            for (int l = 0; l < VEC; ++l) { va[l] = vcentre(g, 0, (int)(e0 + l)); vb[l] = vcentre(g, 2, jz); }
        }
        const double *k = p.K + cell * 12 + 4 * dim;
        const double k0 = __ldg(k), k1 = __ldg(k + 1), ka = __ldg(k + 2), kb = __ldg(k + 3);
        sB = k1 * g.dv[dim];
#pragma unroll
        for (int l = 0; l < VEC; ++l) sA[l] = fma(kb, vb[l], fma(ka, va[l], fma(k1, g.vlo[dim], k0)));
    }

    T buf[U];                                        // g_{i+2} for the next U steps
#pragma unroll
    for (int u = 0; u < U; ++u)
        if (2 + u < n) buf[u] = ldv<VEC>(base + (long long)(2 + u) * inner);
    T w0, w1 = ldv<VEC>(base), w2 = ldv<VEC>(base + inner), w3;
    double pl[VEC];                                  // flux through face i-1/2
#pragma unroll
    for (int l = 0; l < VEC; ++l) { w0.v[l] = 0.0; pl[l] = 0.0; }
    double fi = 1.0;                                 // i + 1 as a double
    for (int i0 = 0; i0 < n; i0 += U) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = i0 + u;
            if (i < n) {
                if (i + 2 < n) w3 = buf[u];
                else {
#pragma unroll
                    for (int l = 0; l < VEC; ++l) w3.v[l] = 0.0;
                }
                if (i + 2 + U < n) buf[u] = ldv<VEC>(base + (long long)(i + 2 + U) * inner);
                T out;
                double sf[VEC], phv[VEC];
#pragma unroll
                for (int l = 0; l < VEC; ++l) sf[l] = fma(fi, sB, sA[l]);
                bs_face_fluxes<VEC>(w0.v, w1.v, w2.v, w3.v, sf, phv);
#pragma unroll
                for (int l = 0; l < VEC; ++l) {
                    const double ph = i == n - 1 ? 0.0 : phv[l];       // closed box (R7)
                    out.v[l] = w1.v[l] + (pl[l] - ph);
                    pl[l] = ph;
                }
                stv<VEC>(base + (long long)i * inner, out);
                w0 = w1; w1 = w2; w2 = w3;
                fi += 1.0;
            }
        }
    }
}

// ---------------------------------------------------------------- contiguous axis vx
// One thread owns CH consecutive cells of a row (nvx % CH == 0): CH + 4 values, CH + 1 faces.
template <int CH>
__global__ void __launch_bounds__(256)
bs_vx_kernel(const BacksubArgs p, long long rows, int rows_per_cta)
{
    const GridDev &g = p.g;
    const int nvx = g.nv[0];
    const int cpr = nvx / CH;
    const int rl = threadIdx.x / cpr;
    const int q = threadIdx.x - rl * cpr;
    const long long row = (long long)blockIdx.x * rows_per_cta + rl;
    const bool active = rl < rows_per_cta && row < rows;
    double w[CH + 4];
    double sA = 0.0, sB = 0.0;
    double *rowp = nullptr;
    if (active) {
        rowp = p.f + row * nvx;
        if (CH == 1) {
#pragma unroll
            for (int m = 0; m < CH + 4; ++m) {
                const int c = q * CH - 2 + m;
                w[m] = (c >= 0 && c < nvx) ? rowp[c] : 0.0;
            }
        } else {                                     // 16-byte loads: the thread's cells and the 2 + 2 cells beside them
            const double2 *p2 = reinterpret_cast<const double2 *>(rowp + q * CH);
#pragma unroll
            for (int m = 0; m < CH / 2 + 2; ++m) {
                const bool in = (m > 0 || q > 0) && (m < CH / 2 + 1 || q + 1 < cpr);
                const double2 t = in ? p2[m - 1] : make_double2(0.0, 0.0);
                w[2 * m] = t.x; w[2 * m + 1] = t.y;
            }
        }
        const long long plane = row / g.nv[1];
        const int jy = (int)(row - plane * g.nv[1]);
        const long long cell = plane / g.nv[2];
        const int jz = (int)(plane - cell * g.nv[2]);
        const double *k = p.K + cell * 12;
        const double k0 = __ldg(k), k1 = __ldg(k + 1), ka = __ldg(k + 2), kb = __ldg(k + 3);
        sB = k1 * g.dv[0];
        // face m of the thread (m = 0..CH) is face (q CH + m) - 1/2 of the row: xi = vlo + (q CH + m) dv
        sA = fma(kb, vcentre(g, 2, jz), fma(ka, vcentre(g, 1, jy), fma(k1, g.vlo[0], k0))) + (double)(q * CH) * sB;
    }
    __syncthreads();                                 // every load of the CTA precedes every store
    if (!active) return;
    double phi[CH + 1];
#pragma unroll
    for (int m = 0; m <= CH; ++m) phi[m] = bs_face_flux(w[m], w[m + 1], w[m + 2], w[m + 3], fma((double)m, sB, sA));
    if (q == 0) phi[0] = 0.0;                        // closed box (R7)
    if (q == cpr - 1) phi[CH] = 0.0;
    if (CH == 1) {
        rowp[q] = w[2] + (phi[0] - phi[1]);
    } else {
#pragma unroll
        for (int m = 0; m < CH; m += 2)
            *reinterpret_cast<double2 *>(rowp + q * CH + m) =
                make_double2(w[m + 2] + (phi[m] - phi[m + 1]), w[m + 3] + (phi[m + 1] - phi[m + 2]));
    }
}

}  // namespace mphv
