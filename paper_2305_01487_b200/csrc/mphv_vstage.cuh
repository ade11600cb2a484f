// mphv_vstage.cuh -- second-generation whole-V-stage kernel: V_vx, V_vy, V_vz (eq. (1), P:L53;
// scheme P:L135, readings R2/R3/R7/R11) and the moments n, j, P (R9/R10) in ONE pass over f.
//
// Same data flow as vcube_kernel (mphv_vcube.cuh) -- TMA plane ring -> V_vx -> shared memory ->
// V_vy -> registers -> V_vz march along the plane stream -> global -- rebuilt around the ncu
// findings of profiles/r01b_f2_ncu_full.md (150 instructions per cell at 48 % issue utilisation):
//   * TWO planes per pipeline iteration: one bulk copy, one split-barrier arrive/wait and one set
//     of loop bookkeeping per 8 cells per thread and stage instead of per 4;
//   * V_vz in march form (one Q per cell; lanes of either sign finish the SAME plane, two planes
//     behind the newest one): no per-lane store-pointer select, no moment correction;
//   * Courant data per thread from a linear form s = a + vz b (a, b per thread and cube), not from
//     shared-memory tables filled by a few threads; E, B read once per cube through the read-only path;
//   * moments with 6 accumulators per thread (sums over the thread's 4 rows weighted 1, m, m^2)
//     instead of 12.
// Requires nvx % 4 == 0, nvy % 4 == 0, nvz even (>= 4); other shapes use vcube_kernel.
#pragma once
#include "mphv_vcube.cuh"
#include "mphv_march.cuh"

namespace mphv {

enum { VS_NXB = 4 };                    // xb pair-buffers (see the hazard note at the stage-A store)

// c1 = (1-|s|)(2-|s|)/6 and -c2 = -(1-|s|)(1+|s|)/6 of a Courant number
__device__ __forceinline__ void courant_poly(double s, double &c1, double &nc2)
{
    const double fr = fabs(s), om = 1.0 - fr;
    c1 = (om * (2.0 - fr)) * (1.0 / 6.0);
    nc2 = (om * (1.0 + fr)) * (-1.0 / 6.0);
}
// the same with 1/6 handed in from the kernel parameters (a constant-bank operand: no immediate moves) and
// t = 1 - |s| reused: c1 = (t/6)(1 + t), -c2 = -(t/6)(2 - t)
__device__ __forceinline__ void courant_poly6(double s, double sixth, double &c1, double &nc2)
{
    const double t = 1.0 - fabs(s), u = t * sixth;
    c1 = u * (1.0 + t);
    nc2 = -u * (2.0 - t);
}

template <int NS, bool MOM, int NVX, int NVY, int TMAX, int MINB>
__global__ void __launch_bounds__(TMAX, MINB)
vstage_kernel(const CubeArgs p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int nvx = NVX > 0 ? NVX : p.nvx, nvy = NVY > 0 ? NVY : p.nvy, nvz = p.nvz;
    const int qx = nvx / 4;
    const int cells = nvx * nvy;
    const int xcells = nvx * (nvy + 4);                                  // xb plane with 2+2 zero rows
    const int hz = nvz / 2;                                              // plane pairs per cube
    const uint32_t pair_bytes = (uint32_t)cells * 16u;
    double *ring = reinterpret_cast<double *>(smem_raw);                 // [NS][2][cells]
    double *xb = ring + (size_t)NS * 2 * cells;                         // [VS_NXB][2][nvy + 4][nvx]
    double *vzt = xb + (size_t)VS_NXB * 2 * xcells;                     // [nvz] vz centres
    double *red = vzt + nvz;                                            // [10][32]
    double2 *zc = reinterpret_cast<double2 *>(red + 320);               // [4][T] V_vz slope coefficients of the thread's pencils
    double *zsm = reinterpret_cast<double *>(zc + 4 * (size_t)blockDim.x);         // [4][T] V_vz Courant numbers of the thread's pencils
    uint64_t *bars = reinterpret_cast<uint64_t *>(zsm + 4 * (size_t)blockDim.x);   // [NS] TMA full, [2] xbar

    const long long c_begin = (p.ns * (long long)blockIdx.x) / gridDim.x;
    const long long c_end = (p.ns * ((long long)blockIdx.x + 1)) / gridDim.x;
    const int ncell = (int)(c_end - c_begin);
    const int K2 = ncell * hz;                                           // plane pairs of this CTA
    if (K2 == 0) return;
    double *const stream0 = p.f + c_begin * (long long)nvz * cells;
    const bool act = tid < nvy * qx;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(&bars[s], 1);
        mbar_init(&bars[NS], (uint32_t)blockDim.x);
        mbar_init(&bars[NS + 1], (uint32_t)blockDim.x);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    for (int i = tid; i < nvz; i += blockDim.x) vzt[i] = vcentre(p.g, 2, i);
    for (int i = tid; i < VS_NXB * 2 * xcells; i += blockDim.x) xb[i] = 0.0;
    __syncthreads();
    if (tid == 0) {
        for (int k = 0; k < NS && k < K2; ++k) {
            mbar_expect_tx(&bars[k], pair_bytes);
            bulk_load(ring + (size_t)k * 2 * cells, stream0 + (size_t)k * 2 * cells, pair_bytes, &bars[k]);
        }
    }

    // thread <-> work
    const int r_x = tid / qx, q_x = tid - r_x * qx;                       // V_vx item: row, quad
    const int rq = tid / nvx, jx = tid - rq * nvx;                        // V_vy / V_vz patch: row quad, column
    const int r0 = 4 * rq;
    const bool xlo_wall = q_x == 0, xhi_wall = q_x == qx - 1;
    const bool ylo_wall = rq == 0, yhi_wall = r0 + 4 == nvy;
    const int in_off = 4 * tid;                                          // doubles, within a ring plane
    const int xw_off = (r_x + 2) * nvx + 4 * q_x;                        // V_vx store, within an xb plane
    const int xr_off = r0 * nvx + jx;                                    // V_vy first row (r0 - 2, + 2 zero rows)
    // (per-thread velocity centres and dt / dv are re-evaluated in the peeled cube-boundary code, so they hold no
    // registers across the iterations inside a cube)

    // per-cube linear forms of the Courant numbers: s = a + vz b
    double ax = 0.0, bx = 0.0, ay = 0.0, by = 0.0;
    // V_vz march state of this thread's 4 pencils (rows r0..r0+3 of column jx)
    // s and the coefficients of lim(g_{j+1}-g_j), lim(g_{j-1}-g_j) live in zsm, zc
    double2 *const zcp = zc + tid;                   // (shared memory, written and read by this thread only)
    double *const zsp = zsm + tid;
    double G0[4], G1[4], Q[4], E[4];                 // the two newest planes (G0: even, G1: odd), Q_i, E_i = Q_{i-1} - Q_i
    double P0 = 0.0, Q1 = 0.0, Q2 = 0.0, Z1 = 0.0, Z2 = 0.0, ZQ = 0.0;   // moment sums (see header)
#pragma unroll
    for (int m = 0; m < 4; ++m) { G0[m] = G1[m] = Q[m] = E[m] = 0.0; }

    // One march step for the 4 pencils: nw = g_{i+2} arrives, Q_{i+1} is formed, cell i is finished
    // and stored to plane i (po). MODE 0: interior; 1: i = nvz-2 (Q_{i+1} sits in front of the high
    // wall); 2: i = nvz-1 (Q_{i+1} is the ghost cell behind it). Closed box, R7.
    // (GA, GB) = (g_i, g_{i+1}) on entry; GA becomes g_{i+2} (the caller alternates the two windows: no rotation)
    auto vz_step = [&](auto mode_tag, double (&GA)[4], double (&GB)[4], const double (&nw)[4], double wz, double *po) {
        constexpr int MODE = decltype(mode_tag)::value;
        double o[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double zs = zsp[m * blockDim.x];
            const bool pos = __double2hiint(zs) >= 0;
            const double2 zxy = zcp[m * blockDim.x];
            double qn = march_q(GA[m], GB[m], nw[m], zxy.x, zxy.y);
            if (MODE == 1 && pos) qn = 0.0;
            if (MODE == 2 && !pos) qn = 0.0;
            const double en = Q[m] - qn;
            o[m] = fma(zs, pos ? E[m] : en, GA[m]);
            Q[m] = qn; E[m] = en;
            GA[m] = nw[m];
            __stcs(po + m * nvx, o[m]);              // streaming store
        }
        if (MOM) {
            const double p0 = (o[0] + o[1]) + (o[2] + o[3]);
            const double q1 = fma(3.0, o[3], fma(2.0, o[2], o[1]));
            const double q2 = fma(9.0, o[3], fma(4.0, o[2], o[1]));
            P0 += p0; Q1 += q1; Q2 += q2;
            const double t = wz * p0;
            Z1 += t; Z2 = fma(wz, t, Z2); ZQ = fma(wz, q1, ZQ);
        }
    };
    struct M0 { enum { value = 0 }; }; struct M1 { enum { value = 1 }; }; struct M2 { enum { value = 2 }; };

    int slotA = 0; uint32_t parA = 0;                // ring slot / phase of pair i (stage A)
    int slotB = 0;                                   // ring slot of pair i-1 (stage B)
    int jA = 0, cellA = 0;                           // (cell, pair in cube) of pair i
    int jB = 0, cellB = 0;                           // (cell, pair in cube) of pair i-1
    double *outp = stream0 + (size_t)r0 * nvx + jx;  // plane 0 of the cube of stage B, this thread's first cell

    // One pipeline iteration: stage A of pair i, stage B of pair i-1. FIRST / LAST: pair i-1 is the first /
    // last pair of its cube (compile-time, so the 18 of 20 iterations in between carry no cube-boundary code).
    // AFIRST: pair i is the first of its cube; HASA: pair i exists (false only in the final call).
    auto iter = [&](auto first_tag, auto last_tag, auto afirst_tag, auto hasa_tag, const int i) {
        constexpr bool FIRST = decltype(first_tag)::value, LAST = decltype(last_tag)::value;
        constexpr bool AFIRST = decltype(afirst_tag)::value, HASA = decltype(hasa_tag)::value;
        // ================= stage A: V_vx of planes 2i, 2i+1
        if (HASA) {
            if (AFIRST) {                            // new cube: a_x = qm (E_x + vy B_z - vz B_y)
                const long long c = c_begin + cellA;
                const double Ex = __ldg(p.E + c), By = __ldg(p.B + p.ns + c), Bz = __ldg(p.B + 2 * p.ns + c);
                const double dtdvx = p.dt / p.g.dv[0], vy_row = vcentre(p.g, 1, act ? r_x : 0);   // a_x needs vy of the row
                ax = (p.g.qm * (Ex + vy_row * Bz)) * dtdvx;
                bx = -(p.g.qm * By) * dtdvx;
            }
            mbar_wait(&bars[slotA], parA);
            if (act) {
                // xb pair-buffer i % 4: last read in stage B of pair i-4 (iteration i-3); every thread
                // left that stage before it arrived for pair i-2, and this thread waited for those
                // arrivals in iteration i-1. Three buffers would not do (pair i-3 is read in iteration
                // i-2, and nothing this thread has waited for orders that before this store).
                double *xdst = xb + (size_t)(i % VS_NXB) * 2 * xcells + xw_off;
                const double *src = ring + (size_t)slotA * 2 * cells + in_off;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const double2 *in2 = reinterpret_cast<const double2 *>(src + h * cells);
                    const double2 o0 = in2[0], o1 = in2[1];
                    double2 l = make_double2(0.0, 0.0), r = make_double2(0.0, 0.0);
                    if (!xlo_wall) l = in2[-1];
                    if (!xhi_wall) r = in2[2];
                    const double w[8] = { l.x, l.y, o0.x, o0.y, o1.x, o1.y, r.x, r.y };
                    const double s = fma(vzt[2 * jA + h], bx, ax);
                    double c1, nc2, o[4];
                    courant_poly6(s, p.sixth, c1, nc2);
                    remap4(w, s, c1, nc2, xlo_wall, xhi_wall, o);
                    double2 *xo = reinterpret_cast<double2 *>(xdst + h * xcells);
                    xo[0] = make_double2(o[0], o[1]);
                    xo[1] = make_double2(o[2], o[3]);
                }
            }
            mbar_arrive(&bars[NS + (i & 1)]);
            slotA = slotA + 1 == NS ? 0 : slotA + 1;
            if (slotA == 0) parA ^= 1u;
            if (++jA == hz) { jA = 0; ++cellA; }
        }
        if (i == 0) return;
        // ================= stage B: V_vy of planes 2(i-1), 2(i-1)+1, two V_vz march steps, moments
        const int ib = i - 1;
        mbar_wait(&bars[NS + (ib & 1)], (uint32_t)((ib >> 1) & 1));
        if (tid == 0 && ib + NS < K2) {              // every thread has consumed ring slot slotB
            mbar_expect_tx(&bars[slotB], pair_bytes);
            bulk_load(ring + (size_t)slotB * 2 * cells, stream0 + (size_t)(ib + NS) * 2 * cells, pair_bytes, &bars[slotB]);
        }
        slotB = slotB + 1 == NS ? 0 : slotB + 1;
        if (FIRST) {                                 // new cube
            const long long c = c_begin + cellB;
            const double Ey = __ldg(p.E + p.ns + c), Ez = __ldg(p.E + 2 * p.ns + c);
            const double Bx = __ldg(p.B + c), By = __ldg(p.B + p.ns + c), Bz = __ldg(p.B + 2 * p.ns + c);
            // a_y = qm (E_y + vz B_x - vx B_z);  a_z = qm (E_z + vx B_y - vy B_x)
            const double dtdvy = p.dt / p.g.dv[1], dtdvz = p.dt / p.g.dv[2], dvy = p.g.dv[1];
            const double vx_col = vcentre(p.g, 0, jx), vy0 = vcentre(p.g, 1, act ? r0 : 0);
            ay = (p.g.qm * (Ey - vx_col * Bz)) * dtdvy;
            by = (p.g.qm * Bx) * dtdvy;
            const double az0 = Ez + vx_col * By;
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                const double s = (p.g.qm * (az0 - fma((double)m, dvy, vy0) * Bx)) * dtdvz;
                double c1, nc2;
                courant_poly(s, c1, nc2);
                const bool pos = __double2hiint(s) >= 0;
                zsp[m * blockDim.x] = s;
                zcp[m * blockDim.x] = pos ? make_double2(c1, nc2) : make_double2(nc2, c1);
            }
            P0 = Q1 = Q2 = Z1 = Z2 = ZQ = 0.0;
        }
        if (act) {
            const double *xsrc = xb + (size_t)(ib % VS_NXB) * 2 * xcells + xr_off;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int jz = 2 * jB + h;
                const double s = fma(vzt[jz], by, ay);
                double c1, nc2, nw[4];
                courant_poly6(s, p.sixth, c1, nc2);
                // the 7-row window starts one row later for s < 0: lanes of either sign run the same code
                const bool pos = __double2hiint(s) >= 0;
                const double *xi = xsrc + h * xcells;
                const double *xw = pos ? xi : xi + nvx;
                const double ccx = pos ? c1 : nc2, ccy = pos ? nc2 : c1;
                double w[7], q[5];
#pragma unroll
                for (int r = 0; r < 7; ++r) w[r] = xw[r * nvx];
#pragma unroll
                for (int r = 0; r < 5; ++r) q[r] = march_q(w[r], w[r + 1], w[r + 2], ccx, ccy);
                if (ylo_wall) q[0] = 0.0;            // closed box (R7): the wall faces carry no flux
                if (yhi_wall) q[4] = 0.0;
#pragma unroll
                for (int r = 0; r < 4; ++r) nw[r] = fma(s, q[r] - q[r + 1], xi[(r + 2) * nvx]);
                if (FIRST) {
                    if (h == 0) {
#pragma unroll
                        for (int m = 0; m < 4; ++m) G0[m] = nw[m];       // g_0
                    } else {
#pragma unroll
                        for (int m = 0; m < 4; ++m) {                    // g_1: Q_0, E_0 (face -1/2 carries no flux)
                            const bool pos = __double2hiint(zsp[m * blockDim.x]) >= 0;
                            G1[m] = nw[m];
                            const double2 zxy = zcp[m * blockDim.x];
                            double q0 = march_q(0.0, G0[m], G1[m], zxy.x, zxy.y);
                            if (!pos) q0 = 0.0;
                            Q[m] = q0; E[m] = -q0;
                        }
                    }
                } else {
                    if (h == 0) vz_step(M0(), G0, G1, nw, vzt[jz - 2], outp);
                    else        vz_step(M0(), G1, G0, nw, vzt[jz - 2], outp);
                    outp += cells;
                }
            }
            if (LAST) {                              // drain: the two ghost planes behind the high wall are empty
                const double zero[4] = { 0.0, 0.0, 0.0, 0.0 };
                vz_step(M1(), G0, G1, zero, vzt[nvz - 2], outp);
                outp += cells;
                vz_step(M2(), G1, G0, zero, vzt[nvz - 1], outp);
                outp += cells;
            }
        }
        if (LAST) {
            if (MOM) {
                double mom[10];
#pragma unroll
                for (int k = 0; k < 10; ++k) mom[k] = 0.0;
                if (act) {
                    // sums over the thread's rows m = 0..3: vy = vy0 + m dvy
                    const double dvy = p.g.dv[1], vx_col = vcentre(p.g, 0, jx), vy0 = vcentre(p.g, 1, r0);
                    const double Sy = fma(dvy, Q1, vy0 * P0);                                    // sum vy f
                    const double Syy = fma(dvy * dvy, Q2, fma(2.0 * vy0 * dvy, Q1, vy0 * vy0 * P0));
                    const double Syz = fma(dvy, ZQ, vy0 * Z1);
                    const double vx = vx_col;
                    mom[0] = P0;
                    mom[1] = vx * P0; mom[2] = Sy; mom[3] = Z1;
                    mom[4] = vx * (vx * P0); mom[5] = vx * Sy; mom[6] = vx * Z1;
                    mom[7] = Syy; mom[8] = Syz; mom[9] = Z2;
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
            jB = 0; ++cellB;
        } else {
            ++jB;
        }
    };
    struct No { enum { value = 0 }; }; struct Yes { enum { value = 1 }; };
    iter(No(), No(), Yes(), Yes(), 0);
    int i = 1;
    for (int cell = 0; cell < ncell; ++cell) {
        iter(Yes(), No(), No(), Yes(), i++);
        for (int j = 1; j < hz - 1; ++j) iter(No(), No(), No(), Yes(), i++);
        if (cell + 1 < ncell) iter(No(), Yes(), Yes(), Yes(), i++);
        else                  iter(No(), Yes(), No(), No(), i++);
    }
}

}  // namespace mphv
