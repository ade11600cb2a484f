// mphv_vstage3.cuh -- fourth-generation whole-V-stage kernel: V_vx, V_vy, V_vz (eq. (1); scheme P:L135,
// readings R2/R3/R7/R11) and the moments n, j, P (R9/R10) in ONE pass over f, WARP-SPECIALISED.
//
// vstage2_kernel (mphv_vstage2.cuh) runs both stages of the pipeline on the same 10 warps: every warp does V_vx of
// plane pair i ("stage A"), then V_vy + V_vz + moments of pair i-1 ("stage B"). The round-2 ncu capture (r02a, git history) and
// profiles/r02_issue_rate.md: it is bound by the latency of each warp's own instruction stream (2.5 warps per
// scheduler, 50 % issue and 52 % fp64-pipe utilisation, 15 % of the warp time in the two barrier waits); stage B
// alone takes 1.53 ms of its 2.17 ms, stage A alone 0.89 ms. Here the two stages run on DIFFERENT warps at the
// same time:
//   B warps (0 .. TB/32-1)   stage B only; their V_vz state lives in registers as before;
//   A warps (TB/32 .. )      stage A only: one run of CH cells of one row per thread and plane pair;
//   last warp, lane 0        the TMA producer: refills a ring slot as soon as the A warps have released it.
// The stages are coupled by mbarrier pairs (full / empty) per ring slot and per xb buffer instead of a CTA-wide
// barrier, so neither waits for the other unless it is a whole buffer ahead. The register file is re-divided with
// setmaxnreg (sm_90a+): the warpgroups that hold B warps take RB registers per thread, the last warpgroup (A warps
// and the producer) keeps RA; A warps that share a warpgroup with B warps run the same code under the larger budget.
// Shapes: NVX % CH == 0, CH even, NVY % P == 0, nvz even and >= 4, TB = (NVY / P) NVX a multiple of 32,
// 2 NVY (NVX / CH) A threads. Other shapes use vstage2_kernel / vstage_kernel.
#pragma once
#include "mphv_vstage2.cuh"

namespace mphv {

__device__ __forceinline__ void named_bar_sync(int id, int threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

template <int NS, bool MOM, int NVX, int NVY, int P, int CH, int TB, int TMAX, int RB, int RA>
__global__ void __launch_bounds__(TMAX, 1)
vstage3_kernel(const CubeArgs p)
{
    constexpr int QX = NVX / CH;                     // V_vx runs per row
    constexpr int CPP = NVY * QX;                    // ... per plane
    constexpr int TA = 2 * CPP;                      // stage-A threads: one run of each plane of the pair
    constexpr int RG = NVY / P;                      // row groups
    constexpr int cells = NVX * NVY;
    constexpr int xcells = NVX * (NVY + 4);          // xb plane with 2 + 2 zero rows
    constexpr int NWB = TB / 32;
    constexpr int NXB = 4;                           // xb pair-buffers
    static_assert(NVX % CH == 0 && CH % 2 == 0 && NVY % P == 0 && TB == RG * NVX && TB % 32 == 0 && NWB <= 16, "shape");
    static_assert(TMAX % 128 == 0 && TB + TA + 32 <= TMAX && TA % 32 == 0, "warp roles");
    static_assert(TB <= TMAX - 128, "the last warpgroup holds no B warp");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int nvz = p.nvz, hz = nvz / 2;             // plane pairs per cube
    constexpr uint32_t pair_bytes = (uint32_t)cells * 16u;
    double *ring = reinterpret_cast<double *>(smem_raw);                 // [NS][2][cells]
    double *xb = ring + (size_t)NS * 2 * cells;                         // [NXB][2][NVY + 4][NVX]
    double *vzt = xb + (size_t)NXB * 2 * xcells;                        // [nvz] vz centres
    double *red = vzt + nvz;                                            // [2][10][16] warp partials of the moments
    uint64_t *tfull = reinterpret_cast<uint64_t *>(red + 320);          // [NS] TMA landed
    uint64_t *tempty = tfull + NS;                                      // [NS] ring slot read by every A thread
    uint64_t *xfull = tempty + NS;                                      // [NXB] xb pair written by every A thread
    uint64_t *xempty = xfull + NXB;                                     // [NXB] xb pair read by every B thread

    const long long c_begin = (p.ns * (long long)blockIdx.x) / gridDim.x;
    const long long c_end = (p.ns * ((long long)blockIdx.x + 1)) / gridDim.x;
    const int ncell = (int)(c_end - c_begin);
    const int K2 = ncell * hz;                                           // plane pairs of this CTA
    if (K2 == 0) return;
    double *const stream0 = p.f + c_begin * (long long)nvz * cells;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], (uint32_t)TA); }
        for (int s = 0; s < NXB; ++s) { mbar_init(&xfull[s], (uint32_t)TA); mbar_init(&xempty[s], (uint32_t)TB); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    for (int i = tid; i < nvz; i += TMAX) vzt[i] = vcentre(p.g, 2, i);
    for (int i = tid; i < NXB * 2 * xcells; i += TMAX) xb[i] = 0.0;
    __syncthreads();

    // ---- re-divide the register file between the roles (every warp of a warpgroup executes its instruction)
    const bool last_wg = tid >= TMAX - 128;
    if (last_wg) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(RA));
    else         asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(RB));

    // ======================================================================================= TMA producer
    if (tid == TMAX - 32) {
        for (int k = 0; k < K2; ++k) {
            const int slot = k % NS;
            if (k >= NS) mbar_wait(&tempty[slot], (uint32_t)((k / NS - 1) & 1));
            mbar_expect_tx(&tfull[slot], pair_bytes);
            bulk_load(ring + (size_t)slot * 2 * cells, stream0 + (size_t)k * 2 * cells, pair_bytes, &tfull[slot]);
        }
        return;
    }
    if (tid >= TB + TA) return;                      // the producer's other lanes, spare warps

    // ======================================================================================= stage A: V_vx
    auto stage_a = [&]() {
        const int ta = tid - TB;                     // run ta of the pair: plane h, row r, run q of the row
        const int h = ta / CPP, cc = ta - h * CPP;
        const int r = cc / QX, q = cc - r * QX;
        const bool xlo_wall = q == 0, xhi_wall = q == QX - 1;
        const int in_off = h * cells + cc * CH;      // doubles within a ring pair
        const int out_off = h * xcells + (r + 2) * NVX + q * CH;
        const double vy_row = vcentre(p.g, 1, r);
        const double dtdvx = p.dt / p.g.dv[0];
        double ax = 0.0, bx = 0.0;                   // per-cube linear form of the Courant number: s = ax + vz bx
        int jA = 0, cellA = 0;
        for (int i = 0; i < K2; ++i) {
            if (jA == 0) {                           // new cube: a_x = qm (E_x + vy B_z - vz B_y)
                const long long c = c_begin + cellA;
                const double Ex = __ldg(p.E + c), By = __ldg(p.B + p.ns + c), Bz = __ldg(p.B + 2 * p.ns + c);
                ax = (p.g.qm * (Ex + vy_row * Bz)) * dtdvx;
                bx = -(p.g.qm * By) * dtdvx;
            }
            const int slot = i % NS, xs = i % NXB;
            const double s = fma(vzt[2 * jA + h], bx, ax);
            double c1, nc2;
            courant_poly6(s, p.sixth, c1, nc2);
            mbar_wait(&tfull[slot], (uint32_t)((i / NS) & 1));
            const double2 *in2 = reinterpret_cast<const double2 *>(ring + (size_t)slot * 2 * cells + in_off);
            if (i >= NXB) mbar_wait(&xempty[xs], (uint32_t)((i / NXB - 1) & 1));
            double2 *xo = reinterpret_cast<double2 *>(xb + (size_t)xs * 2 * xcells + out_off);
            // The run in chunks of 4 cells, loads just ahead of their use (few live registers: this code runs under
            // the small register budget). W[j] = cell j - 2 of the run; pair k = (W[2k], W[2k+1]) = in2[k - 1];
            // q[m] = Q behind face m - 1/2: from cells (m-2, m-1, m) for s >= 0, (m-1, m, m+1) for s < 0.
            const bool pos = __double2hiint(s) >= 0;
            const double cx = pos ? c1 : nc2, cy = pos ? nc2 : c1;
            double W[CH + 4];
            auto load_pair = [&](int k) {
                double2 t = make_double2(0.0, 0.0);
                if (!((k == 0 && xlo_wall) || (k == CH / 2 + 1 && xhi_wall))) t = in2[k - 1];
                W[2 * k] = t.x; W[2 * k + 1] = t.y;
            };
#pragma unroll
            for (int k = 0; k < 4; ++k) load_pair(k);
            double qprev = pos ? march_q(W[0], W[1], W[2], cx, cy) : march_q(W[1], W[2], W[3], cx, cy);
            if (xlo_wall) qprev = 0.0;
#pragma unroll
            for (int t = 0; t < CH / 4; ++t) {
                if (t > 0) { load_pair(2 * t + 2); load_pair(2 * t + 3); }
                double q[5], o[4];
                q[0] = qprev;
#pragma unroll
                for (int m = 1; m <= 4; ++m) {
                    const int j = 4 * t + m;
                    q[m] = pos ? march_q(W[j], W[j + 1], W[j + 2], cx, cy) : march_q(W[j + 1], W[j + 2], W[j + 3], cx, cy);
                }
                if (t == CH / 4 - 1 && xhi_wall) q[4] = 0.0;
#pragma unroll
                for (int m = 0; m < 4; ++m) o[m] = fma(s, q[m] - q[m + 1], W[4 * t + m + 2]);
                xo[2 * t] = make_double2(o[0], o[1]);
                xo[2 * t + 1] = make_double2(o[2], o[3]);
                qprev = q[4];
            }
            mbar_arrive(&tempty[slot]);              // the slot has been read
            mbar_arrive(&xfull[xs]);
            if (++jA == hz) { jA = 0; ++cellA; }
        }
    };
    if (tid >= TB) {
        stage_a();
        return;
    }

    // ======================================================================================= stage B: V_vy, V_vz, moments
    const int rg = tid / NVX, jx = tid - rg * NVX;
    const int r0 = P * rg;
    const bool ylo_wall = rg == 0, yhi_wall = rg == RG - 1;
    const int xr_off = r0 * NVX + jx;                                    // V_vy first row (r0 - 2, + 2 zero rows)
    double ay = 0.0, by = 0.0;                       // per-cube linear form of the V_vy Courant number
    double zs[P], zx[P], zy[P];                      // V_vz: Courant number and slope coefficients of the P pencils
    double G0[P], G1[P], Q[P], E[P];                 // the two newest planes (G0: even, G1: odd), Q_i, E_i = Q_{i-1} - Q_i
    double P0 = 0.0, Q1 = 0.0, Q2 = 0.0, Z1 = 0.0, Z2 = 0.0, ZQ = 0.0;   // moment sums
#pragma unroll
    for (int m = 0; m < P; ++m) { zs[m] = zx[m] = zy[m] = 0.0; G0[m] = G1[m] = Q[m] = E[m] = 0.0; }

    // One march step of the P pencils (see vstage2_kernel): nw = g_{i+2} arrives, Q_{i+1} is formed, cell i is
    // finished and stored to plane i (po). MODE 0: interior; 1: i = nvz-2; 2: i = nvz-1. Closed box, R7.
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

    // Sum of the warp partials of cube `cube` (fixed order) -> global. Without a barrier when the cube has enough
    // pairs: a B warp that has been handed pair i + NXB + 1 knows every B warp has released pair i + 1 (the A warps
    // refill an xb buffer only after all B threads arrived on its empty barrier), hence finished pair i entirely.
    const bool defer = hz >= NXB + 3;
    auto finish_moments = [&](int cube) {
        if (MOM && tid < 10) {
            const double *rr = red + (cube & 1) * 160 + tid * 16;
            double s = rr[0];
#pragma unroll
            for (int w = 1; w < NWB; ++w) s += rr[w];
            const long long cell = c_begin + cube;
            double *dst = tid == 0 ? p.n + cell : tid < 4 ? p.j + (tid - 1) * p.ns + cell : p.P + (tid - 4) * p.ns + cell;
            *dst = s * p.dV;
        }
    };
    int jB = 0, cellB = 0;                           // (cell, pair in cube) of the pair in work
    double *outp = stream0 + (size_t)r0 * NVX + jx;  // plane 0 of the cube, this thread's first cell

    // One pair. FIRST / LAST: it is the first / last pair of its cube (compile-time: the pairs in between carry
    // no cube-boundary code).
    auto pair = [&](auto first_tag, auto last_tag, const int ib) {
        constexpr bool FIRST = decltype(first_tag)::value, LAST = decltype(last_tag)::value;
        if (FIRST) {                                 // new cube
            const long long c = c_begin + cellB;
            const double Ey = __ldg(p.E + p.ns + c), Ez = __ldg(p.E + 2 * p.ns + c);
            const double Bx = __ldg(p.B + c), By = __ldg(p.B + p.ns + c), Bz = __ldg(p.B + 2 * p.ns + c);
            // a_y = qm (E_y + vz B_x - vx B_z);  a_z = qm (E_z + vx B_y - vy B_x)
            const double dtdvy = p.dt / p.g.dv[1], dtdvz = p.dt / p.g.dv[2], dvy = p.g.dv[1];
            const double vx_col = vcentre(p.g, 0, jx), vy0 = vcentre(p.g, 1, r0);
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
        const int xs = ib % NXB;
        mbar_wait(&xfull[xs], (uint32_t)((ib / NXB) & 1));
        if (MOM && !FIRST && !LAST && defer && jB == NXB + 1 && cellB > 0) finish_moments(cellB - 1);
        const double *xsrc = xb + (size_t)xs * 2 * xcells + xr_off;
        double nwp[2][P];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int jz = 2 * jB + h;
            const double s = fma(vzt[jz], by, ay);
            double c1, nc2;
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
            if (ylo_wall) q[0] = 0.0;                // closed box (R7): the wall faces carry no flux
            if (yhi_wall) q[P] = 0.0;
#pragma unroll
            for (int r = 0; r < P; ++r) nwp[h][r] = fma(s, q[r] - q[r + 1], xi[(r + 2) * NVX]);
        }
        mbar_arrive(&xempty[xs]);                    // the xb pair is in registers
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int jz = 2 * jB + h;
            if (FIRST) {
                if (h == 0) {
#pragma unroll
                    for (int m = 0; m < P; ++m) G0[m] = nwp[0][m];      // g_0
                } else {
#pragma unroll
                    for (int m = 0; m < P; ++m) {                        // g_1: Q_0, E_0 (face -1/2 carries no flux)
                        const bool zpos = __double2hiint(zs[m]) >= 0;
                        G1[m] = nwp[1][m];
                        double q0 = march_q(0.0, G0[m], G1[m], zx[m], zy[m]);
                        if (!zpos) q0 = 0.0;
                        Q[m] = q0; E[m] = -q0;
                    }
                }
            } else {
                if (h == 0) vz_step(M0(), G0, G1, nwp[0], vzt[jz - 2], outp);
                else        vz_step(M0(), G1, G0, nwp[1], vzt[jz - 2], outp);
                outp += cells;
            }
        }
        if (LAST) {                                  // drain: the two ghost planes behind the high wall are empty
            double zero[P];
#pragma unroll
            for (int m = 0; m < P; ++m) zero[m] = 0.0;
            vz_step(M1(), G0, G1, zero, vzt[nvz - 2], outp);
            outp += cells;
            vz_step(M2(), G1, G0, zero, vzt[nvz - 1], outp);
            outp += cells;
            if (MOM) {
                // sums over the thread's rows m = 0..P-1: vy = vy0 + m dvy
                const double dvy = p.g.dv[1], vx = vcentre(p.g, 0, jx), vy0 = vcentre(p.g, 1, r0);
                const double Sy = fma(dvy, Q1, vy0 * P0);                                    // sum vy f
                const double Syy = fma(dvy * dvy, Q2, fma(2.0 * vy0 * dvy, Q1, vy0 * vy0 * P0));
                const double Syz = fma(dvy, ZQ, vy0 * Z1);
                const double mom[10] = { P0, vx * P0, Sy, Z1, vx * (vx * P0), vx * Sy, vx * Z1, Syy, Syz, Z2 };
                double *r = red + (cellB & 1) * 160 + (tid >> 5);
#pragma unroll
                for (int k = 0; k < 10; ++k) {
                    double x = mom[k];
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
                    if ((tid & 31) == 0) r[k * 16] = x;
                }
                if (!defer) { named_bar_sync(1, TB); finish_moments(cellB); }   // few pairs per cube: finish at once
            }
            jB = 0; ++cellB;
        } else {
            ++jB;
        }
    };
    struct No { enum { value = 0 }; }; struct Yes { enum { value = 1 }; };
    int ib = 0;
    for (int cell = 0; cell < ncell; ++cell) {
        pair(Yes(), No(), ib++);
        for (int j = 1; j < hz - 1; ++j) pair(No(), No(), ib++);
        pair(No(), Yes(), ib++);
    }
    if (MOM && defer) { named_bar_sync(1, TB); finish_moments(ncell - 1); }
}

}  // namespace mphv
