// mphv_vstage_bs.cuh -- the whole V stage in BACKSUBSTITUTION mode (reading R15, mphv_backsub.cuh) and
// the moments in ONE pass over f: the pipeline of vstage_kernel (TMA plane-pair ring -> V_vx -> shared memory ->
// V_vy -> registers -> V_vz march along the plane stream -> global; split barrier; cube-boundary iterations
// peeled at compile time) with the three sweeps in FACE form: every face has its own Courant number
//     s_face = K0 + K1 xi + Ka va + Kb vb     (the 12 numbers K per spatial cell from backsub_coeff_kernel),
// i.e. per thread and plane an affine sequence s_m = s_0 + m s_B over the thread's 5 faces (V_vx, V_vy) and per
// pencil an affine sequence along the march (V_vz, state: g_{i-1}, g_i, g_{i+1} and the flux through face i-1/2).
// Requires nvx % 4 == 0, nvy % 4 == 0, nvz even (>= 4); other shapes use the three bs_* sweep kernels.
#pragma once
#include "mphv_vstage.cuh"
#include "mphv_backsub.cuh"

namespace mphv {

template <int NS, bool MOM, int NVX, int NVY, int TMAX, int MINB>
__global__ void __launch_bounds__(TMAX, MINB)
vstage_bs_kernel(const CubeArgs p)
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
    const double vy_row = vcentre(p.g, 1, act ? r_x : 0);                // V_vx: a_x needs vy of the row
    const double vx_col = vcentre(p.g, 0, jx);                           // V_vy: a_y needs vx of the column
    const double vy0 = vcentre(p.g, 1, act ? r0 : 0), dvy = p.g.dv[1];

    // per-cube linear forms of the Courant numbers: s = a + vz b
    double ax = 0.0, bx = 0.0, sBx = 0.0, ay = 0.0, by = 0.0, sBy = 0.0, sBz = 0.0;
    // V_vz march state of this thread's 4 pencils (rows r0..r0+3 of column jx)
    // the constant part of each pencil's face Courant number lives in zsm (shared memory, this thread's slots only)
    double *const zsp = zsm + tid;
    double W0[4], W1[4], W2[4], PL[4];               // g_{i-1}, g_i, g_{i+1}, flux through face i-1/2
    double P0 = 0.0, Q1 = 0.0, Q2 = 0.0, Z1 = 0.0, Z2 = 0.0, ZQ = 0.0;   // moment sums (see header)
#pragma unroll
    for (int m = 0; m < 4; ++m) { W0[m] = W1[m] = W2[m] = PL[m] = 0.0; }

    // One march step for the 4 pencils in face form: nw = g_{i+2} arrives, the flux through face i+1/2 (Courant
    // number zsp[m] + fi sBz, fi = i + 1) is formed, cell i is finished and stored to plane i (po).
    // MODE 0: interior (and i = nvz-2, where nw is the empty ghost plane); 2: i = nvz-1, the wall face carries
    // no flux (R7).
    auto vz_step = [&](auto mode_tag, const double (&nw)[4], double fi, double wz, double *po) {
        constexpr int MODE = decltype(mode_tag)::value;
        double o[4], phv[4] = { 0.0, 0.0, 0.0, 0.0 };
        if (MODE != 2) {
            double sf[4];
#pragma unroll
            for (int m = 0; m < 4; ++m) sf[m] = fma(fi, sBz, zsp[m * blockDim.x]);
            bs_face_fluxes<4>(W0, W1, W2, nw, sf, phv);
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double ph = phv[m];
            o[m] = W1[m] + (PL[m] - ph);
            PL[m] = ph;
            W0[m] = W1[m]; W1[m] = W2[m]; W2[m] = nw[m];
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
            if (AFIRST) {                            // new cube: s of the thread's first face = ax + vz bx; next faces + sBx
                const double *k = p.K + (c_begin + cellA) * 12;
                const double k0 = __ldg(k), k1 = __ldg(k + 1), ka = __ldg(k + 2), kb = __ldg(k + 3);
                sBx = k1 * p.g.dv[0];
                ax = fma(ka, vy_row, fma(k1, p.g.vlo[0], k0)) + (double)(4 * q_x) * sBx;
                bx = kb;
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
                    const double s0 = fma(vzt[2 * jA + h], bx, ax);
                    double phi[5], o[4];
#pragma unroll
                    for (int m = 0; m < 5; ++m) phi[m] = bs_face_flux(w[m], w[m + 1], w[m + 2], w[m + 3], fma((double)m, sBx, s0));
                    if (xlo_wall) phi[0] = 0.0;      // closed box (R7)
                    if (xhi_wall) phi[4] = 0.0;
#pragma unroll
                    for (int c = 0; c < 4; ++c) o[c] = w[2 + c] + (phi[c] - phi[c + 1]);
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
        if (FIRST) {                                 // new cube: affine Courant data of V_vy (per plane) and V_vz (per pencil)
            const double *k = p.K + (c_begin + cellB) * 12;
            const double y0 = __ldg(k + 4), y1 = __ldg(k + 5), ya = __ldg(k + 6), yb = __ldg(k + 7);
            const double z0 = __ldg(k + 8), z1 = __ldg(k + 9), za = __ldg(k + 10), zb = __ldg(k + 11);
            // V_vy: face m of the thread (between rows r0-1+m and r0+m) at xi = vlo_y + (r0 + m) dvy; (va, vb) = (vx, vz)
            sBy = y1 * dvy;
            ay = fma(ya, vx_col, fma(y1, p.g.vlo[1], y0)) + (double)r0 * sBy;
            by = yb;
            // V_vz: face i+1/2 at xi = vlo_z + (i + 1) dvz; (va, vb) = (vx, vy of the pencil)
            sBz = z1 * p.g.dv[2];
#pragma unroll
            for (int m = 0; m < 4; ++m)
                zsp[m * blockDim.x] = fma(zb, fma((double)m, dvy, vy0), fma(za, vx_col, fma(z1, p.g.vlo[2], z0)));
            P0 = Q1 = Q2 = Z1 = Z2 = ZQ = 0.0;
        }
        if (act) {
            const double *xsrc = xb + (size_t)(ib % VS_NXB) * 2 * xcells + xr_off;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int jz = 2 * jB + h;
                const double s0 = fma(vzt[jz], by, ay);
                const double *xi = xsrc + h * xcells;
                double w[8], phi[5], nw[4];
#pragma unroll
                for (int r = 0; r < 8; ++r) w[r] = xi[r * nvx];
                {   // the faces of a warp almost always move the same way: select-free upwind paths
                    const double s4 = fma(4.0, sBy, s0);
                    const bool apos = __double2hiint(s0) >= 0 && __double2hiint(s4) >= 0;
                    const bool aneg = __double2hiint(s0) < 0 && __double2hiint(s4) < 0;
                    const unsigned mask = __activemask();
                    if (__all_sync(mask, apos)) {
#pragma unroll
                        for (int m = 0; m < 5; ++m) {
                            const double sm = fma((double)m, sBy, s0), fr = fabs(sm), om = 1.0 - fr;
                            phi[m] = face_flux(w[m], w[m + 1], w[m + 2], sm, (om * (2.0 - fr)) * (1.0 / 6.0), (om * (1.0 + fr)) * (1.0 / 6.0));
                        }
                    } else if (__all_sync(mask, aneg)) {
#pragma unroll
                        for (int m = 0; m < 5; ++m) {
                            const double sm = fma((double)m, sBy, s0), fr = fabs(sm), om = 1.0 - fr;
                            phi[m] = face_flux(w[m + 3], w[m + 2], w[m + 1], sm, (om * (2.0 - fr)) * (1.0 / 6.0), (om * (1.0 + fr)) * (1.0 / 6.0));
                        }
                    } else {
#pragma unroll
                        for (int m = 0; m < 5; ++m) phi[m] = bs_face_flux(w[m], w[m + 1], w[m + 2], w[m + 3], fma((double)m, sBy, s0));
                    }
                }
                if (ylo_wall) phi[0] = 0.0;          // closed box (R7): the wall faces carry no flux
                if (yhi_wall) phi[4] = 0.0;
#pragma unroll
                for (int r = 0; r < 4; ++r) nw[r] = w[2 + r] + (phi[r] - phi[r + 1]);
                if (FIRST) {
                    if (h == 0) {
#pragma unroll
                        for (int m = 0; m < 4; ++m) { W0[m] = 0.0; W1[m] = nw[m]; PL[m] = 0.0; }   // g_0; face -1/2 is the wall
                    } else {
#pragma unroll
                        for (int m = 0; m < 4; ++m) W2[m] = nw[m];                                 // g_1
                    }
                } else {
                    vz_step(M0(), nw, (double)(jz - 1), vzt[jz - 2], outp);
                    outp += cells;
                }
            }
            if (LAST) {                              // drain: the two ghost planes behind the high wall are empty
                const double zero[4] = { 0.0, 0.0, 0.0, 0.0 };
                vz_step(M0(), zero, (double)(nvz - 1), vzt[nvz - 2], outp);
                outp += cells;
                vz_step(M2(), zero, (double)nvz, vzt[nvz - 1], outp);
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
