// mphv_vstage3_bs.cuh -- the whole V stage in BACKSUBSTITUTION mode (reading R15, mphv_backsub.cuh) and the
// moments in ONE pass over f, WARP-SPECIALISED: the roles, buffers, mbarrier protocol and register split of
// vstage3_kernel (mphv_vstage3.cuh) with the three sweeps in FACE form as in vstage_bs_kernel (mphv_vstage_bs.cuh):
// every face has its own Courant number
//     s_face = K0 + K1 xi + Ka va + Kb vb     (the 12 numbers K per spatial cell from backsub_coeff_kernel),
// i.e. per thread and plane an affine sequence s_m = s_0 + m s_B over the faces of its run (V_vx) or patch (V_vy)
// and per pencil an affine sequence along the march (V_vz; state g_{i-1}, g_i, g_{i+1}, the flux through face
// i-1/2 and the constant part of the face Courant number: 5 doubles per pencil, in registers).
// Shapes as vstage3_kernel; other shapes use vstage_bs_kernel or the three bs_* sweep kernels.
#pragma once
#include "mphv_vstage3.cuh"
#include "mphv_backsub.cuh"

namespace mphv {

template <int NS, bool MOM, int NVX, int NVY, int P, int CH, int TB, int TMAX, int RB, int RA>
__global__ void __launch_bounds__(TMAX, 1)
vstage3_bs_kernel(const CubeArgs p)
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
        double ax = 0.0, bx = 0.0, sBx = 0.0;        // per cube: s of the run's face m = ax + vz bx + m sBx
        int jA = 0, cellA = 0;
        for (int i = 0; i < K2; ++i) {
            if (jA == 0) {                           // new cube: face m of the run at xi = vlo_x + (q CH + m) dvx; (va, vb) = (vy, vz)
                const double *k = p.K + (c_begin + cellA) * 12;
                const double k0 = __ldg(k), k1 = __ldg(k + 1), ka = __ldg(k + 2), kb = __ldg(k + 3);
                sBx = k1 * p.g.dv[0];
                ax = fma(ka, vy_row, fma(k1, p.g.vlo[0], k0)) + (double)(q * CH) * sBx;
                bx = kb;
            }
            const int slot = i % NS, xs = i % NXB;
            const double s0 = fma(vzt[2 * jA + h], bx, ax);
            mbar_wait(&tfull[slot], (uint32_t)((i / NS) & 1));
            const double2 *in2 = reinterpret_cast<const double2 *>(ring + (size_t)slot * 2 * cells + in_off);
            if (i >= NXB) mbar_wait(&xempty[xs], (uint32_t)((i / NXB - 1) & 1));
            double2 *xo = reinterpret_cast<double2 *>(xb + (size_t)xs * 2 * xcells + out_off);
            // The run in chunks of 4 cells, loads just ahead of their use (few live registers: this code runs under
            // the small register budget). W[j] = cell j - 2 of the run; pair k = (W[2k], W[2k+1]) = in2[k - 1];
            // face m (between cells m - 1 and m) sees W[m .. m+3] and moves by s0 + m sBx.
            double W[CH + 4];
            auto load_pair = [&](int k) {
                double2 t = make_double2(0.0, 0.0);
                if (!((k == 0 && xlo_wall) || (k == CH / 2 + 1 && xhi_wall))) t = in2[k - 1];
                W[2 * k] = t.x; W[2 * k + 1] = t.y;
            };
#pragma unroll
            for (int k = 0; k < 4; ++k) load_pair(k);
            double phprev = xlo_wall ? 0.0 : bs_face_flux(W[0], W[1], W[2], W[3], s0);     // closed box (R7)
#pragma unroll
            for (int t = 0; t < CH / 4; ++t) {
                if (t > 0) { load_pair(2 * t + 2); load_pair(2 * t + 3); }
                double ph[5], o[4];
                ph[0] = phprev;
#pragma unroll
                for (int m = 1; m <= 4; ++m) {
                    const int j = 4 * t + m;
                    ph[m] = bs_face_flux(W[j], W[j + 1], W[j + 2], W[j + 3], fma((double)j, sBx, s0));
                }
                if (t == CH / 4 - 1 && xhi_wall) ph[4] = 0.0;
#pragma unroll
                for (int m = 0; m < 4; ++m) o[m] = W[4 * t + m + 2] + (ph[m] - ph[m + 1]);
                xo[2 * t] = make_double2(o[0], o[1]);
                xo[2 * t + 1] = make_double2(o[2], o[3]);
                phprev = ph[4];
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
    const double vx_col = vcentre(p.g, 0, jx);       // V_vy: a_y needs vx of the column
    const double vy0 = vcentre(p.g, 1, r0), dvy = p.g.dv[1];
    double ay = 0.0, by = 0.0, sBy = 0.0, sBz = 0.0; // per cube: V_vy face m of the patch moves by ay + vz by + m sBy
    double zc[P];                                    // V_vz: constant part of each pencil's face Courant number
    double W0[P], W1[P], W2[P], PL[P];               // g_{i-1}, g_i, g_{i+1}, flux through face i-1/2
    double P0 = 0.0, Q1 = 0.0, Q2 = 0.0, Z1 = 0.0, Z2 = 0.0, ZQ = 0.0;   // moment sums
#pragma unroll
    for (int m = 0; m < P; ++m) { zc[m] = 0.0; W0[m] = W1[m] = W2[m] = PL[m] = 0.0; }

    // One march step of the P pencils in face form: nw = g_{i+2} arrives, the flux through face i+1/2 (Courant
    // number zc[m] + fi sBz, fi = i + 1) is formed, cell i is finished and stored to plane i (po).
    // MODE 0: interior (and i = nvz-2, where nw is the empty ghost plane); 2: i = nvz-1, the wall face carries
    // no flux (R7).
    auto vz_step = [&](auto mode_tag, const double (&nw)[P], double fi, double wz, double *po) {
        constexpr int MODE = decltype(mode_tag)::value;
        double o[P], phv[P];
#pragma unroll
        for (int m = 0; m < P; ++m) phv[m] = 0.0;
        if (MODE != 2) {
            double sf[P];
#pragma unroll
            for (int m = 0; m < P; ++m) sf[m] = fma(fi, sBz, zc[m]);
            bs_face_fluxes<P>(W0, W1, W2, nw, sf, phv);
        }
#pragma unroll
        for (int m = 0; m < P; ++m) {
            const double ph = phv[m];
            o[m] = W1[m] + (PL[m] - ph);
            PL[m] = ph;
            W0[m] = W1[m]; W1[m] = W2[m]; W2[m] = nw[m];
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
        if (FIRST) {                                 // new cube: affine Courant data of V_vy (per plane) and V_vz (per pencil)
            const double *k = p.K + (c_begin + cellB) * 12;
            const double y0 = __ldg(k + 4), y1 = __ldg(k + 5), ya = __ldg(k + 6), yb = __ldg(k + 7);
            const double z0 = __ldg(k + 8), z1 = __ldg(k + 9), za = __ldg(k + 10), zb = __ldg(k + 11);
            // V_vy: face m of the patch (between rows r0-1+m and r0+m) at xi = vlo_y + (r0 + m) dvy; (va, vb) = (vx, vz)
            sBy = y1 * dvy;
            ay = fma(ya, vx_col, fma(y1, p.g.vlo[1], y0)) + (double)r0 * sBy;
            by = yb;
            // V_vz: face i+1/2 at xi = vlo_z + (i + 1) dvz; (va, vb) = (vx, vy of the pencil)
            sBz = z1 * p.g.dv[2];
#pragma unroll
            for (int m = 0; m < P; ++m)
                zc[m] = fma(zb, fma((double)m, dvy, vy0), fma(za, vx_col, fma(z1, p.g.vlo[2], z0)));
            P0 = Q1 = Q2 = Z1 = Z2 = ZQ = 0.0;
        }
        const int xs = ib % NXB;
        mbar_wait(&xfull[xs], (uint32_t)((ib / NXB) & 1));
        if (MOM && !FIRST && !LAST && defer && jB == NXB + 1 && cellB > 0) finish_moments(cellB - 1);
        const double *xsrc = xb + (size_t)xs * 2 * xcells + xr_off;
        double nwp[2][P];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double s0 = fma(vzt[2 * jB + h], by, ay);
            const double *xi = xsrc + h * xcells;
            double w[P + 4], phi[P + 1];             // rows r0 - 2 .. r0 + P + 1: face m sees w[m .. m + 3]
#pragma unroll
            for (int r = 0; r < P + 4; ++r) w[r] = xi[r * NVX];
            {   // the faces of a warp almost always move the same way: select-free upwind paths
                const double sP = fma((double)P, sBy, s0);
                const bool apos = __double2hiint(s0) >= 0 && __double2hiint(sP) >= 0;
                const bool aneg = __double2hiint(s0) < 0 && __double2hiint(sP) < 0;
                if (__all_sync(0xffffffffu, apos)) {
#pragma unroll
                    for (int m = 0; m <= P; ++m) {
                        const double sm = fma((double)m, sBy, s0), fr = fabs(sm), om = 1.0 - fr;
                        phi[m] = face_flux(w[m], w[m + 1], w[m + 2], sm, (om * (2.0 - fr)) * (1.0 / 6.0), (om * (1.0 + fr)) * (1.0 / 6.0));
                    }
                } else if (__all_sync(0xffffffffu, aneg)) {
#pragma unroll
                    for (int m = 0; m <= P; ++m) {
                        const double sm = fma((double)m, sBy, s0), fr = fabs(sm), om = 1.0 - fr;
                        phi[m] = face_flux(w[m + 3], w[m + 2], w[m + 1], sm, (om * (2.0 - fr)) * (1.0 / 6.0), (om * (1.0 + fr)) * (1.0 / 6.0));
                    }
                } else {
#pragma unroll
                    for (int m = 0; m <= P; ++m) phi[m] = bs_face_flux(w[m], w[m + 1], w[m + 2], w[m + 3], fma((double)m, sBy, s0));
                }
            }
            if (ylo_wall) phi[0] = 0.0;              // closed box (R7): the wall faces carry no flux
            if (yhi_wall) phi[P] = 0.0;
#pragma unroll
            for (int r = 0; r < P; ++r) nwp[h][r] = w[2 + r] + (phi[r] - phi[r + 1]);
        }
        mbar_arrive(&xempty[xs]);                    // the xb pair is in registers
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int jz = 2 * jB + h;
            if (FIRST) {
                if (h == 0) {
#pragma unroll
                    for (int m = 0; m < P; ++m) { W0[m] = 0.0; W1[m] = nwp[0][m]; PL[m] = 0.0; }   // g_0; face -1/2 is the wall
                } else {
#pragma unroll
                    for (int m = 0; m < P; ++m) W2[m] = nwp[1][m];                                 // g_1
                }
            } else {
                vz_step(M0(), nwp[h], (double)(jz - 1), vzt[jz - 2], outp);
                outp += cells;
            }
        }
        if (LAST) {                                  // drain: the two ghost planes behind the high wall are empty
            double zero[P];
#pragma unroll
            for (int m = 0; m < P; ++m) zero[m] = 0.0;
            vz_step(M0(), zero, (double)(nvz - 1), vzt[nvz - 2], outp);
            outp += cells;
            vz_step(M2(), zero, (double)nvz, vzt[nvz - 1], outp);
            outp += cells;
            if (MOM) {
                // sums over the thread's rows m = 0..P-1: vy = vy0 + m dvy
                const double vx = vx_col;
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
