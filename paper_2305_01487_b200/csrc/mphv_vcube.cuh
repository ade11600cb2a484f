// mphv_vcube.cuh -- the whole V stage (V_vx, V_vy, V_vz of eq. (1), scheme P:L135) and
// the moments n, j, P in ONE pass over f: f is read once and written once.
//
// The velocity cube of one spatial cell is nvz contiguous planes of nvy x nvx doubles
// (12.8 KB at 40^2). A persistent CTA owns a contiguous range of spatial cells, i.e. one
// contiguous stream of planes:
//   TMA      one bulk async copy (cp.async.bulk, mbarrier completion) per plane into an
//            NS-deep shared-memory ring -- no registers are tied up by loads in flight.
//   V_vx     thread <-> 4 consecutive cells of a row: reads 8 values (2+4+2) from the ring
//            slot, 5 face fluxes, writes 4 new cells to xb[k & 1] (shared memory).
//   barrier  one __syncthreads per plane (xb complete; ring slot free -> next TMA issued).
//   V_vy     thread <-> 4 consecutive rows of one column: reads 8 values from xb, 5 face
//            fluxes, 4 new cells stay in REGISTERS.
//   V_vz     those 4 cells are the newest entries of four register windows marching along
//            vz (the plane stream IS the vz march): cell-based form -- with
//            Q_j = g_j + c1 lim(g_{j+1}-g_j) - c2 lim(g_{j-1}-g_j)   (s >= 0; mirrored for s < 0)
//            the face flux is phi_{j+1/2} = s Q_j (s >= 0) or s Q_{j+1} (s < 0), so
//            new_j = g_j + s (Q_{j-1} - Q_j)  resp.  new_{j-1} = g_{j-1} + s (Q_{j-1} - Q_j):
//            one Q per cell and plane, lanes of either sign run the same code and differ
//            only in which plane they store to.
//   moments  S0 += new, S1 += vz new, S2 += vz^2 new per thread-cell along the march; at the
//            end of the cube combined with vx, vy and block-reduced to the 10 moments.
// Limited slopes (R2), division-free: lim(d, b) = (d > 0 && 2b < d) ? 2b : d, evaluated as
// (max(2b, 0) < d) ? 2b : d  (identical for every finite input, one compare per slope).
#pragma once
#include "mphv_kernels.cuh"

namespace mphv {

struct CubeArgs {
    double *f;
    long long ns;           // spatial cells
    int nvx, nvy, nvz;
    int qx;                 // nvx / 4: vx items per row
    int items;              // nvy * qx == (nvy / 4) * nvx: active threads
    double dt;
    const double *E, *B;
    double *n, *j, *P;      // MOM only
    double dV;
    GridDev g;
};

__device__ __forceinline__ double lim_slope(double d, double cap, double capp)
{
    return (capp < d) ? cap : d;
}

// Q of the cell with value b, downwind neighbour c, upwind neighbour a (uniform-sign form:
// for s < 0 the caller swaps a and c, which is the mirror image, R11).
__device__ __forceinline__ double cell_q(double a, double b, double c, double c1, double c2)
{
    const double cap = b + b;
    const double capp = (__double2hiint(cap) < 0) ? 0.0 : cap;      // max(cap, +0)
    const double lp = lim_slope(c - b, cap, capp);
    const double lm = lim_slope(a - b, cap, capp);                  // = -L^-
    return fma(-c2, lm, fma(c1, lp, b));
}

// 4 new cells from 8 consecutive values w (cells -2 .. 5 relative to the first owned cell)
// along an axis with uniform Courant data (sf, c1, c2); wall_lo / wall_hi close the box (R7).
__device__ __forceinline__ void remap4(const double (&w)[8], double sf, double c1, double c2,
                                       bool wall_lo, bool wall_hi, double (&out)[4])
{
    double q[5];                                     // Q behind faces -1/2 .. 7/2
    if (sf >= 0.0) {
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = cell_q(w[m], w[m + 1], w[m + 2], c1, c2);
    } else {
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = cell_q(w[m + 3], w[m + 2], w[m + 1], c1, c2);
    }
    if (wall_lo) q[0] = 0.0;
    if (wall_hi) q[4] = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) out[c] = fma(sf, q[c] - q[c + 1], w[2 + c]);
}

template <int NS, bool MOM>
__global__ void __launch_bounds__(512, 1)
vcube_kernel(const CubeArgs p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int nvx = p.nvx, nvy = p.nvy, nvz = p.nvz;
    const int cells = nvx * nvy;
    const uint32_t plane_bytes = (uint32_t)cells * 8u;
    double *inbuf = reinterpret_cast<double *>(smem_raw);                // [NS][cells]
    double *xb = inbuf + (size_t)NS * cells;                            // [2][cells]
    double *tabx = xb + 2 * (size_t)cells;                              // [3][3][nvy] row Courant data
    double *taby = tabx + 9 * nvy;                                      // [3][3][nvx] column Courant data
    double *vzt = taby + 9 * nvx;                                       // [nvz + 2] vz centres (index + 1)
    double *fld = vzt + nvz + 2;                                        // [2][6] E, B of this / the next cell
    double *red = fld + 12;                                             // [10][32]
    uint64_t *bars = reinterpret_cast<uint64_t *>(red + 320);           // [NS]

    const long long c_begin = (p.ns * (long long)blockIdx.x) / gridDim.x;
    const long long c_end = (p.ns * ((long long)blockIdx.x + 1)) / gridDim.x;
    const long long K = (c_end - c_begin) * nvz;                         // planes of this CTA
    if (K == 0) return;
    const double *stream0 = p.f + c_begin * (long long)nvz * cells;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(&bars[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (tid < nvz + 2) vzt[tid] = (tid >= 1 && tid <= nvz) ? vcentre(p.g, 2, tid - 1) : 0.0;
    if (tid < 6) fld[tid] = (tid < 3 ? p.E : p.B)[(tid % 3) * p.ns + c_begin];
    __syncthreads();
    if (tid == 0) {
        for (int k = 0; k < NS && k < K; ++k) {
            mbar_expect_tx(&bars[k], plane_bytes);
            bulk_load(inbuf + (size_t)k * cells, stream0 + (long long)k * cells, plane_bytes, &bars[k]);
        }
    }

    const bool act = tid < p.items;
    const int r_x = tid / p.qx, q_x = tid - r_x * p.qx;                   // vx item: row, quad
    const int rq = tid / nvx, jx = tid - rq * nvx;                        // vy/vz patch: row quad, column
    const int r0 = 4 * rq;
    const bool xlo_wall = q_x == 0, xhi_wall = q_x == p.qx - 1;
    const bool ylo_wall = rq == 0, yhi_wall = r0 + 4 == nvy;

    // Courant data of plane (cell, jz) -> table buffer tb: rows (a_x from vy, vz), columns (a_y from vz, vx)
    auto fill_tables = [&](int tb, const double *fl, int jz) {
        if (tid < nvy) {
            const double a = accel(p.g.qm, fl[0], fl[4], fl[5], vcentre(p.g, 1, tid), vzt[jz + 1]);
            const Courant c = make_courant(__ddiv_rn(__dmul_rn(a, p.dt), p.g.dv[0]));
            double *t = tabx + tb * 3 * nvy;
            t[tid] = c.sf; t[nvy + tid] = c.c1; t[2 * nvy + tid] = c.c2;
        } else if (tid < nvy + nvx) {
            const int c0 = tid - nvy;
            const double a = accel(p.g.qm, fl[1], fl[5], fl[3], vzt[jz + 1], vcentre(p.g, 0, c0));
            const Courant c = make_courant(__ddiv_rn(__dmul_rn(a, p.dt), p.g.dv[1]));
            double *t = taby + tb * 3 * nvx;
            t[c0] = c.sf; t[nvx + c0] = c.c1; t[2 * nvx + c0] = c.c2;
        }
    };
    fill_tables(0, fld, 0);
    fill_tables(1, fld, 1);
    __syncthreads();

    int slot = 0; uint32_t parity = 0; int tb = 0;                       // ring slot / phase, table buffer of plane k
    long long k = 0;
    for (long long cell = c_begin; cell < c_end; ++cell) {
        const int cpar = (int)((cell - c_begin) & 1);
        const double *fl = fld + 6 * cpar;
        if (tid < 6 && cell + 1 < c_end) fld[6 * (cpar ^ 1) + tid] = (tid < 3 ? p.E : p.B)[(tid % 3) * p.ns + cell + 1];

        // V_vz Courant data of this thread's 4 pencils: a_z = (q/m)(E_z + vx B_y - vy B_x)
        double zs[4], zx[4], zy[4];                  // s, coefficient of lim(g_{j+1}-g_j), of lim(g_{j-1}-g_j)
        int zoff[4];                                 // store offset of the lane: 0 (s >= 0) or one plane back
        if (act) {
            const double vx = vcentre(p.g, 0, jx);
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                const double a = accel(p.g.qm, fl[2], fl[3], fl[4], vx, vcentre(p.g, 1, r0 + m));
                const Courant c = make_courant(__ddiv_rn(__dmul_rn(a, p.dt), p.g.dv[2]));
                zs[m] = c.sf;
                zx[m] = c.pos ? c.c1 : -c.c2;
                zy[m] = c.pos ? -c.c2 : c.c1;
                zoff[m] = c.pos ? 0 : 1;
            }
        }
        double gm[4], g0[4], qp[4];                  // g_{j-1}, g_j, Q_{j-1}
        double s0[4], s1[4], s2 = 0.0;
#pragma unroll
        for (int m = 0; m < 4; ++m) { gm[m] = 0.0; g0[m] = 0.0; qp[m] = 0.0; s0[m] = 0.0; s1[m] = 0.0; }
        double *cube = p.f + cell * (long long)nvz * cells + (long long)r0 * nvx + jx;

        // one step of the four vz marches: g_{j+1} = nw arrives, Q_j is formed, lanes with s >= 0
        // finish cell j, lanes with s < 0 finish cell j-1.
        auto vz_step = [&](int j, const double (&nw)[4]) {
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                const double b = g0[m];
                const double cap = b + b;
                const double capp = (__double2hiint(cap) < 0) ? 0.0 : cap;
                const double lp = lim_slope(nw[m] - b, cap, capp);
                const double lm = lim_slope(gm[m] - b, cap, capp);
                double q = fma(zy[m], lm, fma(zx[m], lp, b));
                // closed box (R7): faces -1/2 and nvz-1/2 carry no flux
                const bool neg = zoff[m] != 0;
                if ((!neg && j == nvz - 1) || (neg && (j == 0 || j == nvz))) q = 0.0;
                const double gsel = neg ? gm[m] : b;
                const double out = fma(zs[m], qp[m] - q, gsel);
                const int jo = j - zoff[m];
                if (jo >= 0 && jo < nvz) {
                    cube[(long long)jo * cells + m * nvx] = out;
                    if (MOM) {
                        const double vz = vzt[jo + 1];
                        const double t = vz * out;
                        s0[m] += out; s1[m] += t; s2 = fma(vz, t, s2);
                    }
                }
                qp[m] = q; gm[m] = b; g0[m] = nw[m];
            }
        };

        for (int jz = 0; jz < nvz; ++jz, ++k) {
            mbar_wait(&bars[slot], parity);
            const int par = (int)(k & 1);
            // ---- V_vx: ring slot -> xb[par]
            if (act) {
                const double2 *in2 = reinterpret_cast<const double2 *>(inbuf + (size_t)slot * cells);
                double2 *xo = reinterpret_cast<double2 *>(xb + (size_t)par * cells);
                const double2 o0 = in2[2 * tid], o1 = in2[2 * tid + 1];
                double2 l = make_double2(0.0, 0.0), r = make_double2(0.0, 0.0);
                if (!xlo_wall) l = in2[2 * tid - 1];
                if (!xhi_wall) r = in2[2 * tid + 2];
                const double w[8] = { l.x, l.y, o0.x, o0.y, o1.x, o1.y, r.x, r.y };
                const double *t = tabx + tb * 3 * nvy;
                double o[4];
                remap4(w, t[r_x], t[nvy + r_x], t[2 * nvy + r_x], xlo_wall, xhi_wall, o);
                xo[2 * tid] = make_double2(o[0], o[1]);
                xo[2 * tid + 1] = make_double2(o[2], o[3]);
            }
            __syncthreads();                         // xb[par] complete; ring slot consumed by every thread
            if (tid == 0 && k + NS < K) {
                mbar_expect_tx(&bars[slot], plane_bytes);
                bulk_load(inbuf + (size_t)slot * cells, stream0 + (k + NS) * cells, plane_bytes, &bars[slot]);
            }
            // Courant tables of plane k+2 (read after the NEXT barrier; buffer last read before this one)
            if (k + 2 < K) {
                const int tb2 = tb == 0 ? 2 : tb - 1;                    // (tb + 2) % 3
                if (jz + 2 < nvz) fill_tables(tb2, fl, jz + 2);
                else fill_tables(tb2, fld + 6 * (cpar ^ 1), jz + 2 - nvz);
            }
            // ---- V_vy: xb[par] -> registers, then one step of the vz marches
            if (act) {
                const double *xi = xb + (size_t)par * cells + jx;
                double w[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int r = r0 - 2 + i;
                    w[i] = (r >= 0 && r < nvy) ? xi[r * nvx] : 0.0;
                }
                const double *t = taby + tb * 3 * nvx;
                double nw[4];
                remap4(w, t[jx], t[nvx + jx], t[2 * nvx + jx], ylo_wall, yhi_wall, nw);
                if (jz == 0) {
#pragma unroll
                    for (int m = 0; m < 4; ++m) g0[m] = nw[m];
                } else {
                    vz_step(jz - 1, nw);
                }
            }
            slot = slot + 1 == NS ? 0 : slot + 1;
            if (slot == 0) parity ^= 1u;
            tb = tb == 2 ? 0 : tb + 1;
        }
        // drain: the two ghost planes behind the high wall are empty
        if (act) {
            const double zero[4] = { 0.0, 0.0, 0.0, 0.0 };
            vz_step(nvz - 1, zero);
            vz_step(nvz, zero);
        }
        if (MOM) {
            double mom[10];
#pragma unroll
            for (int i = 0; i < 10; ++i) mom[i] = 0.0;
            if (act) {
                const double vx = vcentre(p.g, 0, jx);
#pragma unroll
                for (int m = 0; m < 4; ++m) {
                    const double vy = vcentre(p.g, 1, r0 + m);
                    const double x0 = vx * s0[m], y0 = vy * s0[m];
                    mom[0] += s0[m];
                    mom[1] += x0; mom[2] += y0; mom[3] += s1[m];
                    mom[4] = fma(vx, x0, mom[4]); mom[5] = fma(vx, y0, mom[5]); mom[6] = fma(vx, s1[m], mom[6]);
                    mom[7] = fma(vy, y0, mom[7]); mom[8] = fma(vy, s1[m], mom[8]);
                }
                mom[9] = s2;
            }
            block_reduce_sum<10>(mom, red);
            if (tid == 0) {
                p.n[cell] = mom[0] * p.dV;
#pragma unroll
                for (int a = 0; a < 3; ++a) p.j[a * p.ns + cell] = mom[1 + a] * p.dV;
#pragma unroll
                for (int a = 0; a < 6; ++a) p.P[a * p.ns + cell] = mom[4 + a] * p.dV;
            }
        }
    }
}

}  // namespace mphv
