// mphv_vstage2.cuh -- third-generation whole-V-stage kernel: V_vx, V_vy, V_vz (eq. (1); scheme P:L135,
// readings R2/R3/R7/R11) and the moments n, j, P (R9/R10) in ONE pass over f.
//
// Same data flow as vstage_kernel (mphv_vstage.cuh): TMA ring of plane pairs -> V_vx -> shared memory ->
// V_vy -> registers -> V_vz march along the plane stream -> global, split barrier between the two stages.
// Rebuilt around what profiles/r02_issue_rate.md and the round-1 ncu capture (r01g, git history) show: the warps of that kernel
// are latency-bound (6 cycles per executed instruction per warp, 3.25 warps per scheduler at the 128-register
// cap of a 13-warp CTA), so time follows the instructions one warp executes per plane pair. Here
//   * the work items are LONGER and the CTA SMALLER: V_vx on runs of CH consecutive cells (CH + 1 cell fluxes
//     for CH cells, not 5 for 4), V_vy / V_vz on patches of P rows of one column (P + 1 for P); 40 x 40 planes
//     take P = 5, CH = 10: 320 threads = 10 full warps (no idle lanes), at most 3 warps per scheduler, so up
//     to 168 registers per thread;
//   * with those registers the V_vz Courant numbers and slope coefficients of the thread's P pencils stay in
//     registers (vstage_kernel re-read them from shared memory at every march step);
//   * the moments of a cube are reduced without a CTA-wide barrier: warp partials go to shared memory and ten
//     threads finish the sum two pipeline iterations later, behind the stage barrier they wait on anyway.
// Shapes: NVX % CH == 0, CH even, NVY % P == 0, nvz even and >= 4. Other shapes use vstage_kernel / vcube_kernel.
#pragma once
#include "mphv_vstage.cuh"

namespace mphv {

// CH new cells from CH + 4 consecutive values w (cells -2 .. CH+1 relative to the first owned cell) along an
// axis with uniform Courant data (s, c1, -c2); wall_lo / wall_hi close the box (R7).
template <int CH>
__device__ __forceinline__ void remap_run(const double (&w)[CH + 4], double s, double c1, double nc2,
                                          bool wall_lo, bool wall_hi, double (&out)[CH])
{
    double q[CH + 1];                                // q[m] = Q behind face m - 1/2
    if (s >= 0.0) {
#pragma unroll
        for (int m = 0; m <= CH; ++m) q[m] = march_q(w[m], w[m + 1], w[m + 2], c1, nc2);
    } else {
#pragma unroll
        for (int m = 0; m <= CH; ++m) q[m] = march_q(w[m + 1], w[m + 2], w[m + 3], nc2, c1);
    }
    if (wall_lo) q[0] = 0.0;
    if (wall_hi) q[CH] = 0.0;
#pragma unroll
    for (int c = 0; c < CH; ++c) out[c] = fma(s, q[c] - q[c + 1], w[2 + c]);
}

// TMAX = threads per CTA (the launch must use exactly TMAX); LB >= TMAX only sets the register budget of
// __launch_bounds__ (a scheduler's register file holds 16384: 3 warps of 32 x 168, not 3 x 204).
template <int NS, bool MOM, int NVX, int NVY, int P, int CH, int TMAX, int LB, int MINB>
__global__ void __launch_bounds__(LB, MINB)
vstage2_kernel(const CubeArgs p)
{
    constexpr int QX = NVX / CH;                     // V_vx runs per row
    constexpr int CPP = NVY * QX;                    // ... per plane
    constexpr int NA = 2 * CPP;                      // ... per plane pair
    constexpr int RA = (NA + TMAX - 1) / TMAX;       // stage-A rounds per thread
    constexpr int RG = NVY / P;                      // row groups
    constexpr int TB = RG * NVX;                     // stage-B threads
    constexpr int cells = NVX * NVY;
    constexpr int xcells = NVX * (NVY + 4);          // xb plane with 2 + 2 zero rows
    constexpr int NW = TMAX / 32;
    static_assert(NVX % CH == 0 && CH % 2 == 0 && NVY % P == 0 && TB <= TMAX && TMAX % 32 == 0 && NW <= 16, "shape");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int nvz = p.nvz, hz = nvz / 2;             // plane pairs per cube
    constexpr uint32_t pair_bytes = (uint32_t)cells * 16u;
    double *ring = reinterpret_cast<double *>(smem_raw);                 // [NS][2][cells]
    double *xb = ring + (size_t)NS * 2 * cells;                         // [VS_NXB][2][NVY + 4][NVX]
    double *vzt = xb + (size_t)VS_NXB * 2 * xcells;                     // [nvz] vz centres
    double *red = vzt + nvz;                                            // [2][10][16] warp partials of the moments
    uint64_t *bars = reinterpret_cast<uint64_t *>(red + 320);           // [NS] TMA full, [2] xbar

    const long long c_begin = (p.ns * (long long)blockIdx.x) / gridDim.x;
    const long long c_end = (p.ns * ((long long)blockIdx.x + 1)) / gridDim.x;
    const int ncell = (int)(c_end - c_begin);
    const int K2 = ncell * hz;                                           // plane pairs of this CTA
    if (K2 == 0) return;
    double *const stream0 = p.f + c_begin * (long long)nvz * cells;
    const bool actB = TB == TMAX || tid < TB;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(&bars[s], 1);
        mbar_init(&bars[NS], (uint32_t)TMAX);
        mbar_init(&bars[NS + 1], (uint32_t)TMAX);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    for (int i = tid; i < nvz; i += TMAX) vzt[i] = vcentre(p.g, 2, i);
    for (int i = tid; i < VS_NXB * 2 * xcells; i += TMAX) xb[i] = 0.0;
    __syncthreads();
    if (tid == 0) {
        for (int k = 0; k < NS && k < K2; ++k) {
            mbar_expect_tx(&bars[k], pair_bytes);
            bulk_load(ring + (size_t)k * 2 * cells, stream0 + (size_t)k * 2 * cells, pair_bytes, &bars[k]);
        }
    }

    // ---- thread <-> work
    // stage A, round k: run c = tid + k TMAX of the pair: plane h, row r, run q of the row
    // stage B: rows r0 .. r0 + P - 1 of column jx
    const int rg = tid / NVX, jx = tid - rg * NVX;
    const int r0 = P * rg;
    const bool ylo_wall = rg == 0, yhi_wall = rg == RG - 1;
    const int xr_off = r0 * NVX + jx;                                    // V_vy first row (r0 - 2, + 2 zero rows)

    double ax[RA], bx = 0.0, ay = 0.0, by = 0.0;     // per-cube linear forms of the Courant numbers: s = a + vz b
#pragma unroll
    for (int k = 0; k < RA; ++k) ax[k] = 0.0;
    double zs[P], zx[P], zy[P];                      // V_vz: Courant number and slope coefficients of the P pencils
    double G0[P], G1[P], Q[P], E[P];                 // the two newest planes (G0: even, G1: odd), Q_i, E_i = Q_{i-1} - Q_i
    double P0 = 0.0, Q1 = 0.0, Q2 = 0.0, Z1 = 0.0, Z2 = 0.0, ZQ = 0.0;   // moment sums
#pragma unroll
    for (int m = 0; m < P; ++m) { zs[m] = zx[m] = zy[m] = 0.0; G0[m] = G1[m] = Q[m] = E[m] = 0.0; }

    // One march step of the P pencils: nw = g_{i+2} arrives, Q_{i+1} is formed, cell i is finished and stored
    // to plane i (po). MODE 0: interior; 1: i = nvz-2 (Q_{i+1} sits in front of the high wall); 2: i = nvz-1
    // (Q_{i+1} is the ghost cell behind it). Closed box, R7. (GA, GB) = (g_i, g_{i+1}) on entry; GA becomes
    // g_{i+2} (the caller alternates the two windows: no rotation).
    auto vz_step = [&](auto mode_tag, double (&GA)[P], double (&GB)[P], const double (&nw)[P], double wz, double *po) {
        constexpr int MODE = decltype(mode_tag)::value;
        double o[P];
#pragma unroll
        for (int m = 0; m < P; ++m) {
            const bool pos = __double2hiint(zs[m]) >= 0;
            double qn = march_q(GA[m], GB[m], nw[m], zx[m], zy[m]);
            if (MODE == 1 && pos) qn = 0.0;
            if (MODE == 2 && !pos) qn = 0.0;
            const double en = Q[m] - qn;
            o[m] = fma(zs[m], pos ? E[m] : en, GA[m]);
            Q[m] = qn; E[m] = en;
            GA[m] = nw[m];
            __stcs(po + m * NVX, o[m]);              // streaming store
        }
        if (MOM) {
            double p0 = o[0], q1 = 0.0, q2 = 0.0;
#pragma unroll
            for (int m = 1; m < P; ++m) {
                p0 += o[m];
                q1 = m == 1 ? o[1] : fma((double)m, o[m], q1);
                q2 = m == 1 ? o[1] : fma((double)(m * m), o[m], q2);
            }
            P0 += p0; Q1 += q1; Q2 += q2;
            const double t = wz * p0;
            Z1 += t; Z2 = fma(wz, t, Z2); ZQ = fma(wz, q1, ZQ);
        }
    };
    struct M0 { enum { value = 0 }; }; struct M1 { enum { value = 1 }; }; struct M2 { enum { value = 2 }; };

    // sum of the warp partials of cube `cube` (fixed order) -> global
    auto finish_moments = [&](int cube) {
        if (MOM && tid < 10) {
            const double *r = red + (cube & 1) * 160 + tid * 16;
            double s = r[0];
#pragma unroll
            for (int w = 1; w < NW; ++w) s += r[w];
            const long long cell = c_begin + cube;
            double *dst = tid == 0 ? p.n + cell : tid < 4 ? p.j + (tid - 1) * p.ns + cell : p.P + (tid - 4) * p.ns + cell;
            *dst = s * p.dV;
        }
    };

    int slotA = 0; uint32_t parA = 0;                // ring slot / phase of pair i (stage A)
    int slotB = 0;                                   // ring slot of pair i-1 (stage B)
    int jA = 0, cellA = 0;                           // (cell, pair in cube) of pair i
    int jB = 0, cellB = 0;                           // (cell, pair in cube) of pair i-1
    double *outp = stream0 + (size_t)r0 * NVX + jx;  // plane 0 of the cube of stage B, this thread's first cell

    // One pipeline iteration: stage A of pair i, stage B of pair i-1. FIRST / LAST: pair i-1 is the first /
    // last pair of its cube (compile-time, so the iterations in between carry no cube-boundary code).
    // AFIRST: pair i is the first of its cube; HASA: pair i exists (false only in the final call).
    auto iter = [&](auto first_tag, auto last_tag, auto afirst_tag, auto hasa_tag, const int i) {
        constexpr bool FIRST = decltype(first_tag)::value, LAST = decltype(last_tag)::value;
        constexpr bool AFIRST = decltype(afirst_tag)::value, HASA = decltype(hasa_tag)::value;
        // ================= stage A: V_vx of planes 2i, 2i+1
        if (HASA) {
            if (AFIRST) {                            // new cube: a_x = qm (E_x + vy B_z - vz B_y)
                const long long c = c_begin + cellA;
                const double Ex = __ldg(p.E + c), By = __ldg(p.B + p.ns + c), Bz = __ldg(p.B + 2 * p.ns + c);
                const double dtdvx = p.dt / p.g.dv[0];
#pragma unroll
                for (int k = 0; k < RA; ++k) {
                    const int cc = (tid + k * TMAX) % CPP;
                    ax[k] = (p.g.qm * (Ex + vcentre(p.g, 1, cc / QX) * Bz)) * dtdvx;
                }
                bx = -(p.g.qm * By) * dtdvx;
            }
            mbar_wait(&bars[slotA], parA);
            // xb pair-buffer i % 4: last read in stage B of pair i-4 (iteration i-3); every thread left that
            // stage before it arrived for pair i-2, and this thread waited for those arrivals in iteration
            // i-1. Three buffers would not do.
            double *const xpair = xb + (size_t)(i % VS_NXB) * 2 * xcells;
            const double *const rpair = ring + (size_t)slotA * 2 * cells;
#pragma unroll
            for (int k = 0; k < RA; ++k) {
                const int c = tid + k * TMAX;
                if (NA % TMAX == 0 || c < NA) {
                    const int h = c / CPP, cc = c - h * CPP;
                    const int r = cc / QX, q = cc - r * QX;
                    const bool xlo_wall = q == 0, xhi_wall = q == QX - 1;
                    const double2 *in2 = reinterpret_cast<const double2 *>(rpair + h * cells + cc * CH);
                    double w[CH + 4];
                    double2 t = make_double2(0.0, 0.0);
                    if (!xlo_wall) t = in2[-1];
                    w[0] = t.x; w[1] = t.y;
#pragma unroll
                    for (int u = 0; u < CH / 2; ++u) { t = in2[u]; w[2 + 2 * u] = t.x; w[3 + 2 * u] = t.y; }
                    t = make_double2(0.0, 0.0);
                    if (!xhi_wall) t = in2[CH / 2];
                    w[CH + 2] = t.x; w[CH + 3] = t.y;
                    const double s = fma(vzt[2 * jA + h], bx, ax[k]);
                    double c1, nc2, o[CH];
                    courant_poly6(s, p.sixth, c1, nc2);
                    remap_run<CH>(w, s, c1, nc2, xlo_wall, xhi_wall, o);
                    double2 *xo = reinterpret_cast<double2 *>(xpair + h * xcells + (r + 2) * NVX + q * CH);
#pragma unroll
                    for (int u = 0; u < CH / 2; ++u) xo[u] = make_double2(o[2 * u], o[2 * u + 1]);
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
        // moments of the previous cube: its warp partials were written in stage B two iterations ago, i.e.
        // before every thread's arrive for pair i-1 -- the arrivals this thread has just waited for
        if (MOM && !FIRST && jB == 1 && cellB > 0) finish_moments(cellB - 1);
        if (FIRST) {                                 // new cube
            const long long c = c_begin + cellB;
            const double Ey = __ldg(p.E + p.ns + c), Ez = __ldg(p.E + 2 * p.ns + c);
            const double Bx = __ldg(p.B + c), By = __ldg(p.B + p.ns + c), Bz = __ldg(p.B + 2 * p.ns + c);
            // a_y = qm (E_y + vz B_x - vx B_z);  a_z = qm (E_z + vx B_y - vy B_x)
            const double dtdvy = p.dt / p.g.dv[1], dtdvz = p.dt / p.g.dv[2], dvy = p.g.dv[1];
            const double vx_col = vcentre(p.g, 0, jx), vy0 = vcentre(p.g, 1, actB ? r0 : 0);
            ay = (p.g.qm * (Ey - vx_col * Bz)) * dtdvy;
            by = (p.g.qm * Bx) * dtdvy;
            const double az0 = Ez + vx_col * By;
#pragma unroll
            for (int m = 0; m < P; ++m) {
                const double s = (p.g.qm * (az0 - fma((double)m, dvy, vy0) * Bx)) * dtdvz;
                double c1, nc2;
                courant_poly(s, c1, nc2);
                const bool pos = __double2hiint(s) >= 0;
                zs[m] = s;
                zx[m] = pos ? c1 : nc2;
                zy[m] = pos ? nc2 : c1;
            }
            P0 = Q1 = Q2 = Z1 = Z2 = ZQ = 0.0;
        }
        if (actB) {
            const double *xsrc = xb + (size_t)(ib % VS_NXB) * 2 * xcells + xr_off;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int jz = 2 * jB + h;
                const double s = fma(vzt[jz], by, ay);
                double c1, nc2, nw[P];
                courant_poly6(s, p.sixth, c1, nc2);
                // the (P + 3)-row window starts one row later for s < 0: lanes of either sign run the same code
                const bool pos = __double2hiint(s) >= 0;
                const double *xi = xsrc + h * xcells;
                const double *xw = pos ? xi : xi + NVX;
                const double ccx = pos ? c1 : nc2, ccy = pos ? nc2 : c1;
                double w[P + 3], q[P + 1];
#pragma unroll
                for (int r = 0; r < P + 3; ++r) w[r] = xw[r * NVX];
#pragma unroll
                for (int r = 0; r <= P; ++r) q[r] = march_q(w[r], w[r + 1], w[r + 2], ccx, ccy);
                if (ylo_wall) q[0] = 0.0;            // closed box (R7): the wall faces carry no flux
                if (yhi_wall) q[P] = 0.0;
#pragma unroll
                for (int r = 0; r < P; ++r) nw[r] = fma(s, q[r] - q[r + 1], xi[(r + 2) * NVX]);
                if (FIRST) {
                    if (h == 0) {
#pragma unroll
                        for (int m = 0; m < P; ++m) G0[m] = nw[m];       // g_0
                    } else {
#pragma unroll
                        for (int m = 0; m < P; ++m) {                    // g_1: Q_0, E_0 (face -1/2 carries no flux)
                            const bool zpos = __double2hiint(zs[m]) >= 0;
                            G1[m] = nw[m];
                            double q0 = march_q(0.0, G0[m], G1[m], zx[m], zy[m]);
                            if (!zpos) q0 = 0.0;
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
                double zero[P];
#pragma unroll
                for (int m = 0; m < P; ++m) zero[m] = 0.0;
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
                if (actB) {
                    // sums over the thread's rows m = 0..P-1: vy = vy0 + m dvy
                    const double dvy = p.g.dv[1], vx = vcentre(p.g, 0, jx), vy0 = vcentre(p.g, 1, r0);
                    const double Sy = fma(dvy, Q1, vy0 * P0);                                    // sum vy f
                    const double Syy = fma(dvy * dvy, Q2, fma(2.0 * vy0 * dvy, Q1, vy0 * vy0 * P0));
                    const double Syz = fma(dvy, ZQ, vy0 * Z1);
                    mom[0] = P0;
                    mom[1] = vx * P0; mom[2] = Sy; mom[3] = Z1;
                    mom[4] = vx * (vx * P0); mom[5] = vx * Sy; mom[6] = vx * Z1;
                    mom[7] = Syy; mom[8] = Syz; mom[9] = Z2;
                }
                double *r = red + (cellB & 1) * 160 + (tid >> 5);
#pragma unroll
                for (int k = 0; k < 10; ++k) {
                    double x = mom[k];
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
                    if ((tid & 31) == 0) r[k * 16] = x;
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
    if (MOM) {
        __syncthreads();
        finish_moments(ncell - 1);
    }
}

}  // namespace mphv
