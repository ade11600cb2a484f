// mphv_vcube.cuh -- the whole V stage (V_vx, V_vy, V_vz of eq. (1), scheme P:L135) and
// the moments n, j, P in ONE pass over f: f is read once and written once.
//
// The velocity cube of one spatial cell is nvz contiguous planes of nvy x nvx doubles
// (12.8 KB at 40^2). A persistent CTA owns a contiguous range of spatial cells, i.e. one
// contiguous stream of planes k = 0 .. K-1, and runs a two-stage software pipeline over it:
//
//   iteration k:   [A]  wait TMA(k);  V_vx(k): ring slot -> xb[k % 4];  arrive(xbar[k & 1])
//                  [B]  wait(xbar[(k-1) & 1]);  refill the ring;  V_vy(k-1): xb -> registers;
//                       one step of the V_vz marches; moments
//
//   TMA      one bulk async copy (cp.async.bulk, mbarrier completion) per plane into an
//            NS-deep shared-memory ring -- no registers are tied up by loads in flight.
//   V_vx     thread <-> 4 consecutive cells of a row: 8 values (2+4+2) from the ring slot,
//            5 cell fluxes, 4 new cells to xb (shared memory, two zero rows above and below).
//   xbar     split barrier (mbarrier arrive ... wait one stage later): between a thread's
//            arrive for plane k and its wait lies stage B of plane k-1, so no warp idles at
//            a block-wide barrier.
//   V_vy     thread <-> 4 consecutive rows of one column: 8 values from xb, 5 cell fluxes,
//            the 4 new cells stay in REGISTERS.
//   V_vz     those 4 cells are the newest entries of four register windows marching along
//            vz (the plane stream IS the vz march). Cell-based form: with
//              Q_j = g_j + c1 lim(g_{j+1}-g_j) - c2 lim(g_{j-1}-g_j)   (s >= 0; mirrored for s < 0)
//            the face flux is phi_{j+1/2} = s Q_j (s >= 0) or s Q_{j+1} (s < 0), hence
//              new_j = g_j + s (Q_{j-1} - Q_j)   resp.   new_{j-1} = g_{j-1} + s (Q_{j-1} - Q_j):
//            one Q per cell and plane; lanes of either sign run the same code and differ
//            only in the plane they store to.
//   moments  S0 += new, S1 += vz new, S2 += vz^2 new per thread-cell along the march (with the
//            plane's vz for every lane; lanes with s < 0, which are one plane behind, are
//            corrected once per cube), combined with vx, vy and block-reduced per cube.
// Limited slopes (R2), division-free: lim(d, b) = (d > 0 && 2b < d) ? 2b : d, evaluated as
// (max(2b, 0) < d) ? 2b : d  (identical for every input, one fp64 compare per slope).
#pragma once
#include "mphv_kernels.cuh"

namespace mphv {

struct CubeArgs {
    double *f;
    long long ns;           // spatial cells
    int nvx, nvy, nvz;
    double dt;
    const double *E, *B;
    double *n, *j, *P;      // MOM only
    double dV;
    double sixth;           // 1/6 as a constant-bank operand
    const double *K;        // backsubstitution mode: [ns][12] face-displacement coefficients (mphv_backsub.cuh)
    GridDev g;
};

enum { CUBE_NXB = 4, CUBE_NT = 6, CUBE_FLD = 64 };   // xb buffers, Courant-table buffers, cells per CTA (max)

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Q of the cell with value b, downwind neighbour c, upwind neighbour a (for s < 0 the caller
// swaps a and c: the mirror image, R11).
__device__ __forceinline__ double cell_q(double a, double b, double c, double c1, double nc2)
{
    const double cap = b + b;
    const double capp = b + fabs(b);                                // max(cap, +0) exactly: 2b for b >= 0, +0 for b < 0 (one DADD, no select)
    const double dp = c - b, dm = a - b;
    const double lp = (capp < dp) ? cap : dp;
    const double lm = (capp < dm) ? cap : dm;                        // = -L^-
    return fma(nc2, lm, fma(c1, lp, b));
}

// 4 new cells from 8 consecutive values w (cells -2 .. 5 relative to the first owned cell)
// along an axis with uniform Courant data (s, c1, -c2); wall_lo / wall_hi close the box (R7).
__device__ __forceinline__ void remap4(const double (&w)[8], double sf, double c1, double nc2,
                                       bool wall_lo, bool wall_hi, double (&out)[4])
{
    double q[5];                                     // Q behind faces -1/2 .. 7/2
    if (sf >= 0.0) {
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = cell_q(w[m], w[m + 1], w[m + 2], c1, nc2);
    } else {
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = cell_q(w[m + 3], w[m + 2], w[m + 1], c1, nc2);
    }
    if (wall_lo) q[0] = 0.0;
    if (wall_hi) q[4] = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) out[c] = fma(sf, q[c] - q[c + 1], w[2 + c]);
}

// Courant data (s, c1, -c2, 0) of one pencil from its acceleration; dtdv = dt / dv
__device__ __forceinline__ void courant_entry(double a, double dtdv, double *dst)
{
    const double s = a * dtdv;
    const double fr = fabs(s), om = 1.0 - fr;
    dst[0] = s;
    dst[1] = (om * (2.0 - fr)) * (1.0 / 6.0);
    dst[2] = -((om * (1.0 + fr)) * (1.0 / 6.0));
    dst[3] = 0.0;
}

// VZ = false: V_vx and V_vy only (the V_vy result is stored straight to global memory; V_vz and the
// moments are left to the march kernel) -- no per-thread march state, so two CTAs fit on an SM.
template <int NS, bool VZ, bool MOM, int NVX, int NVY, int TMAX, int MINB>
__global__ void __launch_bounds__(TMAX, MINB)
vcube_kernel(const CubeArgs p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int nvx = NVX > 0 ? NVX : p.nvx, nvy = NVY > 0 ? NVY : p.nvy, nvz = p.nvz;
    const int qx = nvx / 4;
    const int cells = nvx * nvy;
    const int xcells = nvx * (nvy + 4);                                  // xb buffer with 2+2 zero rows
    const uint32_t plane_bytes = (uint32_t)cells * 8u;
    double *inbuf = reinterpret_cast<double *>(smem_raw);                // [NS][cells]
    double *xb = inbuf + (size_t)NS * cells;                            // [NXB][nvy + 4][nvx]
    double *tabx = xb + (size_t)CUBE_NXB * xcells;                      // [NT][nvy][4] row Courant data
    double *taby = tabx + CUBE_NT * 4 * nvy;                            // [NT][nvx][4] column Courant data
    double *vzt = taby + CUBE_NT * 4 * nvx;                             // [nvz] vz centres
    double *fld = vzt + nvz;                                            // [CUBE_FLD][6] E, B of this CTA's cells
    double *red = fld + 6 * CUBE_FLD;                                   // [10][32] (VZ && MOM only)
    uint64_t *bars = reinterpret_cast<uint64_t *>(red + (VZ && MOM ? 320 : 0));   // [NS] TMA full, [2] xbar

    const long long c_begin = (p.ns * (long long)blockIdx.x) / gridDim.x;
    const long long c_end = (p.ns * ((long long)blockIdx.x + 1)) / gridDim.x;
    const int ncell = (int)(c_end - c_begin);
    const int K = ncell * nvz;                                           // planes of this CTA
    if (K == 0) return;
    double *const stream0 = p.f + c_begin * (long long)nvz * cells;
    const int items = nvy * qx;
    const bool act = tid < items;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(&bars[s], 1);
        mbar_init(&bars[NS], (uint32_t)blockDim.x);
        mbar_init(&bars[NS + 1], (uint32_t)blockDim.x);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    for (int i = tid; i < nvz; i += blockDim.x) vzt[i] = vcentre(p.g, 2, i);
    for (int i = tid; i < 6 * ncell; i += blockDim.x) {
        const int c = i / 6, comp = i - 6 * c;
        fld[i] = (comp < 3 ? p.E : p.B)[(comp % 3) * p.ns + c_begin + c];
    }
    for (int i = tid; i < CUBE_NXB * xcells; i += blockDim.x) xb[i] = 0.0;
    __syncthreads();
    if (tid == 0) {
        for (int k = 0; k < NS && k < K; ++k) {
            mbar_expect_tx(&bars[k], plane_bytes);
            bulk_load(inbuf + (size_t)k * cells, stream0 + (size_t)k * cells, plane_bytes, &bars[k]);
        }
    }

    const double dtdvx = p.dt / p.g.dv[0], dtdvy = p.dt / p.g.dv[1], dtdvz = p.dt / p.g.dv[2];
    // Courant data of plane (c, jz) of this CTA -> table buffer tb: rows (a_x from vy, vz), columns (a_y from vz, vx)
    auto fill_tables = [&](int tb, int c, int jz) {
        const double *fl = fld + 6 * c;
        if (tid < nvy) {
            const double a = accel(p.g.qm, fl[0], fl[4], fl[5], vcentre(p.g, 1, tid), vzt[jz]);
            courant_entry(a, dtdvx, tabx + (tb * nvy + tid) * 4);
        } else if (tid < nvy + nvx) {
            const int c0 = tid - nvy;
            const double a = accel(p.g.qm, fl[1], fl[5], fl[3], vzt[jz], vcentre(p.g, 0, c0));
            courant_entry(a, dtdvy, taby + (tb * nvx + c0) * 4);
        }
    };
    for (int k = 0; k < 4 && k < K; ++k) fill_tables(k, k / nvz, k % nvz);
    __syncthreads();

    // thread <-> work
    const int r_x = tid / qx, q_x = tid - r_x * qx;                       // V_vx item: row, quad
    const int rq = tid / nvx, jx = tid - rq * nvx;                        // V_vy / V_vz patch: row quad, column
    const int r0 = 4 * rq;
    const bool xlo_wall = q_x == 0, xhi_wall = q_x == qx - 1;
    const int in_off = 4 * tid;                                          // doubles, within a ring slot
    const int xw_off = (r_x + 2) * nvx + 4 * q_x;                        // V_vx store, within an xb buffer
    const int xr_off = r0 * nvx + jx;                                    // V_vy first row (r0 - 2, + 2 zero rows)
    const double *const tx_ptr = tabx + r_x * 4;
    const double *const ty_ptr = taby + jx * 4;
    const double dvz = p.g.dv[2];

    // V_vz state of this thread's 4 pencils
    double zs[4], zx[4], zy[4];                      // s, coefficient of lim(g_{j+1}-g_j), of lim(g_{j-1}-g_j)
    double ga[4], gb[4], qp[4];                      // window (roles alternate), Q_{j-1}
    double s0[4], s1[4], s2[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) { zs[m] = zx[m] = zy[m] = 0.0; ga[m] = gb[m] = qp[m] = 0.0; s0[m] = s1[m] = s2[m] = 0.0; }
    double *outp = stream0 + (size_t)r0 * nvx + jx;  // plane j of the current cube, this thread's first cell

    // One step of the four marches. gm = g_{j-1}, g0 = g_j, nw = g_{j+1}; Q_j is formed; lanes with
    // s >= 0 finish cell j, lanes with s < 0 finish cell j-1. MODE 0: 1 <= j <= nvz-2; 1: j = 0;
    // 2: j = nvz-1; 3: j = nvz (closed box, R7: faces -1/2 and nvz-1/2 carry no flux).
    // On return gm holds g_{j+1} (the caller swaps the roles of the two window arrays).
    auto vz_step = [&](auto mode_tag, double (&gm)[4], double (&g0)[4], const double (&nw)[4], double wz, double *po) {
        constexpr int MODE = decltype(mode_tag)::value;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double b = g0[m];
            const bool neg = __double2hiint(zs[m]) < 0;
            double q;
            if (MODE == 3) {
                q = 0.0;
            } else {
                const double cap = b + b;
                const double capp = (__double2hiint(cap) < 0) ? 0.0 : cap;
                const double dp = nw[m] - b, dm = gm[m] - b;
                const double lp = (capp < dp) ? cap : dp;
                const double lm = (capp < dm) ? cap : dm;
                q = fma(zy[m], lm, fma(zx[m], lp, b));
                if (MODE == 1 && neg) q = 0.0;
                if (MODE == 2 && !neg) q = 0.0;
            }
            const double out = fma(zs[m], qp[m] - q, neg ? gm[m] : b);
            const bool st = MODE == 0 || MODE == 2 || (MODE == 1 && !neg) || (MODE == 3 && neg);
            if (st) {
                double *dst = po + m * nvx;
                if (neg) dst -= cells;
                *dst = out;
                if (MOM) {
                    const double t = wz * out;
                    s0[m] += out; s1[m] += t; s2[m] = fma(wz, t, s2[m]);
                }
            }
            qp[m] = q;
            gm[m] = nw[m];
        }
    };
    struct M0 { enum { value = 0 }; }; struct M1 { enum { value = 1 }; };
    struct M2 { enum { value = 2 }; }; struct M3 { enum { value = 3 }; };

    int slotA = 0; uint32_t parA = 0;                // ring slot / phase of plane k (stage A)
    int slotB = 0;                                   // ring slot of plane k-1 (stage B)
    int jzB = 0, cellB = 0;                          // (cell, jz) of plane k-1
    int jzT = 4 % nvz, cellT = 4 / nvz;              // (cell, jz) of plane k+3, whose Courant tables stage B fills
    bool flip = false;                               // which window array is g_{j-1}

    for (int k = 0; k <= K; ++k) {
        // ================= stage A: V_vx of plane k
        if (k < K) {
            mbar_wait(&bars[slotA], parA);
            if (act) {
                const double2 *in2 = reinterpret_cast<const double2 *>(inbuf + (size_t)slotA * cells + in_off);
                const double2 o0 = in2[0], o1 = in2[1];
                double2 l = make_double2(0.0, 0.0), r = make_double2(0.0, 0.0);
                if (!xlo_wall) l = in2[-1];
                if (!xhi_wall) r = in2[2];
                const double w[8] = { l.x, l.y, o0.x, o0.y, o1.x, o1.y, r.x, r.y };
                const double *t = tx_ptr + (k % CUBE_NT) * 4 * nvy;
                const double2 t01 = *reinterpret_cast<const double2 *>(t);
                double o[4];
                remap4(w, t01.x, t01.y, t[2], xlo_wall, xhi_wall, o);
                double2 *xo = reinterpret_cast<double2 *>(xb + (size_t)(k % CUBE_NXB) * xcells + xw_off);
                xo[0] = make_double2(o[0], o[1]);
                xo[1] = make_double2(o[2], o[3]);
            }
            mbar_arrive(&bars[NS + (k & 1)]);
            slotA = slotA + 1 == NS ? 0 : slotA + 1;
            if (slotA == 0) parA ^= 1u;
        }
        if (k == 0) continue;
        // ================= stage B: V_vy of plane k-1, one V_vz step, moments
        const int kb = k - 1;
        mbar_wait(&bars[NS + (kb & 1)], (uint32_t)((kb >> 1) & 1));
        if (tid == 0 && kb + NS < K) {               // every thread has consumed ring slot slotB
            mbar_expect_tx(&bars[slotB], plane_bytes);
            bulk_load(inbuf + (size_t)slotB * cells, stream0 + (size_t)(kb + NS) * cells, plane_bytes, &bars[slotB]);
        }
        slotB = slotB + 1 == NS ? 0 : slotB + 1;
        // Courant tables of plane k+3: first read in stage A of iteration k+3, whose threads have waited
        // for plane k+1, i.e. for this thread's arrive after this fill. The buffer was last read in
        // stage B of plane k+3-NT (iteration k+4-NT <= k-2), which every thread left before it arrived
        // for plane k-1 -- the arrive this thread has just waited for.
        if (kb + 4 < K) {
            fill_tables((kb + 4) % CUBE_NT, cellT, jzT);
            if (++jzT == nvz) { jzT = 0; ++cellT; }
        }
        if (act) {
            if (VZ && jzB == 0) {                    // new cube: V_vz Courant data of the 4 pencils
                const double *fl = fld + 6 * cellB;
                const double vx = vcentre(p.g, 0, jx);
#pragma unroll
                for (int m = 0; m < 4; ++m) {
                    const double a = accel(p.g.qm, fl[2], fl[3], fl[4], vx, vcentre(p.g, 1, r0 + m));
                    double e[4];
                    courant_entry(a, dtdvz, e);
                    const bool pos = __double2hiint(e[0]) >= 0;
                    zs[m] = e[0];
                    zx[m] = pos ? e[1] : e[2];
                    zy[m] = pos ? e[2] : e[1];
                    qp[m] = 0.0; ga[m] = 0.0; gb[m] = 0.0;
                    s0[m] = 0.0; s1[m] = 0.0; s2[m] = 0.0;
                }
                flip = false;
            }
            const double *xi = xb + (size_t)(kb % CUBE_NXB) * xcells + xr_off;
            double w[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) w[i] = xi[i * nvx];
            const double *t = ty_ptr + (kb % CUBE_NT) * 4 * nvx;
            const double2 t01 = *reinterpret_cast<const double2 *>(t);
            double nw[4];
            remap4(w, t01.x, t01.y, t[2], rq == 0, r0 + 4 == nvy, nw);
            if (!VZ) {
#pragma unroll
                for (int m = 0; m < 4; ++m) outp[m * nvx] = nw[m];
                outp += cells;
            } else
            // window roles: !flip: ga = g_{j-1}, gb = g_j; flip: the other way round
            if (jzB == 0) {
#pragma unroll
                for (int m = 0; m < 4; ++m) gb[m] = nw[m];               // g_0; ga = g_{-1} = 0
            } else {
                const double wz = vzt[jzB - 1];
                if (jzB == 1) { if (!flip) vz_step(M1(), ga, gb, nw, wz, outp); else vz_step(M1(), gb, ga, nw, wz, outp); }
                else          { if (!flip) vz_step(M0(), ga, gb, nw, wz, outp); else vz_step(M0(), gb, ga, nw, wz, outp); }
                flip = !flip;
                outp += cells;
            }
            if (VZ && jzB == nvz - 1) {              // drain: the two ghost planes behind the high wall are empty
                const double zero[4] = { 0.0, 0.0, 0.0, 0.0 };
                if (!flip) vz_step(M2(), ga, gb, zero, vzt[nvz - 1], outp); else vz_step(M2(), gb, ga, zero, vzt[nvz - 1], outp);
                flip = !flip;
                outp += cells;
                if (!flip) vz_step(M3(), ga, gb, zero, vzt[nvz - 1] + dvz, outp); else vz_step(M3(), gb, ga, zero, vzt[nvz - 1] + dvz, outp);
            }
        }
        if (jzB == nvz - 1) {
            if (VZ && MOM) {
                double mom[10];
#pragma unroll
                for (int i = 0; i < 10; ++i) mom[i] = 0.0;
                if (act) {
                    const double vx = vcentre(p.g, 0, jx);
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        double a0 = s0[m], a1 = s1[m], a2 = s2[m];
                        if (__double2hiint(zs[m]) < 0) {                 // stored one plane behind: vz -> vz - dvz
                            a2 = fma(dvz, fma(dvz, a0, -2.0 * a1), a2);
                            a1 = fma(-dvz, a0, a1);
                        }
                        const double vy = vcentre(p.g, 1, r0 + m);
                        const double x0 = vx * a0, y0 = vy * a0;
                        mom[0] += a0;
                        mom[1] += x0; mom[2] += y0; mom[3] += a1;
                        mom[4] = fma(vx, x0, mom[4]); mom[5] = fma(vx, y0, mom[5]); mom[6] = fma(vx, a1, mom[6]);
                        mom[7] = fma(vy, y0, mom[7]); mom[8] = fma(vy, a1, mom[8]); mom[9] += a2;
                    }
                }
                block_reduce_sum<10>(mom, red);
                if (tid == 0) {
                    const long long cell = c_begin + cellB;
                    p.n[cell] = mom[0] * p.dV;
#pragma unroll
                    for (int a = 0; a < 3; ++a) p.j[a * p.ns + cell] = mom[1 + a] * p.dV;
#pragma unroll
                    for (int a = 0; a < 6; ++a) p.P[a * p.ns + cell] = mom[4 + a] * p.dV;
                }
            }
            jzB = 0; ++cellB;
        } else {
            ++jzB;
        }
    }
}

}  // namespace mphv
