// mphv_march.cuh -- 1-D PFC-3 remap along a STRIDED axis (x, y, z, vy, vz), in place, |s| < 1.
//
// One thread owns VEC adjacent pencils (adjacent in the contiguous index: one double2) and marches
// along the axis; a warp touches 32*VEC*8 contiguous bytes per march step, so stride-N directions
// stay coalesced without a transpose.
//
// Cell-based form of the scheme (R2, R3, R11). With lim(d, b) = (d > 0 && 2b < d) ? 2b : d and
//     Q_j = g_j + c1 lim(g_{j+1}-g_j, g_j) - c2 lim(g_{j-1}-g_j, g_j)      for s >= 0
//     Q_j = g_j + c1 lim(g_{j-1}-g_j, g_j) - c2 lim(g_{j+1}-g_j, g_j)      for s <  0
// the face flux is phi_{j+1/2} = s Q_j (s >= 0) or s Q_{j+1} (s < 0), so with E_j = Q_{j-1} - Q_j
//     new_i = g_i + s E_i   (s >= 0),        new_i = g_i + s E_{i+1}   (s < 0):
// ONE Q per cell, identical code for lanes of either sign (the sign only swaps two per-pencil
// coefficients and picks E_i or E_{i+1}), no per-face selects of the stencil values.
//
// Loop structure: loads run U steps ahead in a ping-pong register buffer (2 x U independent
// 16-byte loads per thread in flight); the main loop has no bounds checks -- (n - 2) mod 2U
// steps are peeled in front of it, the two steps that need ghost cells behind it.
#pragma once
#include "mphv_kernels.cuh"

namespace mphv {

// Q of a cell (value b, lower neighbour a, upper neighbour c) with per-pencil coefficients
// cx (of the upper slope) and cy (of the lower slope): (c1, -c2) for s >= 0, (-c2, c1) for s < 0.
__device__ __forceinline__ double march_q(double a, double b, double c, double cx, double cy)
{
    const double cap = b + b;
    const double capp = b + fabs(b);                                // max(cap, +0) exactly: 2b for b >= 0, +0 for b < 0 (one DADD, no select)
    const double dp = c - b, dm = a - b;
    const double lp = (capp < dp) ? cap : dp;
    const double lm = (capp < dm) ? cap : dm;
    return fma(cy, lm, fma(cx, lp, b));
}

// N cell fluxes Q_m = march_q(w[m], w[m+1], w[m+2]) (STRIDE 1: sliding window) or
// march_q(a[m], b[m], c[m]) with a WARP-UNIFORM fast path: "the limiter only for small values of the
// phase space distribution function" -- where no lane of the warp has a slope above twice its
// cell value (cap >= d+ and cap >= d- everywhere), lim(d) = d and Q = b + cx d+ + cy d- needs no
// select at all (bitwise the same result: the slow path evaluates the same two fma with lp = d+, lm = d-).
template <int N>
__device__ __forceinline__ void march_q_window(const double *w, double cx, double cy, double *q)
{
    double dp[N], dm[N];
    bool plain = true;
#pragma unroll
    for (int m = 0; m < N; ++m) {
        const double b = w[m + 1], cap = b + b;
        dp[m] = w[m + 2] - b; dm[m] = w[m] - b;
        plain = plain && !(cap < dp[m]) && !(cap < dm[m]);
    }
    if (__all_sync(__activemask(), plain)) {
#pragma unroll
        for (int m = 0; m < N; ++m) q[m] = fma(cy, dm[m], fma(cx, dp[m], w[m + 1]));
    } else {
#pragma unroll
        for (int m = 0; m < N; ++m) q[m] = march_q(w[m], w[m + 1], w[m + 2], cx, cy);
    }
}
template <int N>
__device__ __forceinline__ void march_q_lanes(const double *a, const double *b, const double *c,
                                              double cx, double cy, double *q)
{
    double dp[N], dm[N];
    bool plain = true;
#pragma unroll
    for (int m = 0; m < N; ++m) {
        const double cap = b[m] + b[m];
        dp[m] = c[m] - b[m]; dm[m] = a[m] - b[m];
        plain = plain && !(cap < dp[m]) && !(cap < dm[m]);
    }
    if (__all_sync(__activemask(), plain)) {
#pragma unroll
        for (int m = 0; m < N; ++m) q[m] = fma(cy, dm[m], fma(cx, dp[m], b[m]));
    } else {
#pragma unroll
        for (int m = 0; m < N; ++m) q[m] = march_q(a[m], b[m], c[m], cx, cy);
    }
}

template <int VEC, int U, int KIND, int BC, bool MOM, int MINB>
__global__ void __launch_bounds__(256, MINB)
march2_kernel(const MarchArgs p)
{
    typedef V<VEC> T;
    __shared__ double red[MOM ? 10 * 32 : 1];
    const long long innerV = p.inner / VEC;
    long long o, ev;
    bool active;
    if (MOM) {
        // CTA-tiled: blockIdx.x = o * tiles + tile, a CTA never straddles spatial cells
        o = blockIdx.x / p.tiles;
        const int tile = blockIdx.x - (int)o * p.tiles;
        const int lt = threadIdx.x;
        ev = (long long)tile * p.per_tile + lt;
        active = lt < p.per_tile && ev < innerV;
    } else {
        const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        active = t < p.outer * innerV;
        o = t / innerV;
        ev = t - o * innerV;
        if (!active) return;
    }
    double mom[10];
    if (MOM) {
#pragma unroll
        for (int k = 0; k < 10; ++k) mom[k] = 0.0;
    }
    if (active) {
        const long long e0 = ev * VEC;
        const int n = p.n;
        const long long stride = p.inner;
        double *base = p.f + (o * n) * stride + e0;

        double sf[VEC], cx[VEC], cy[VEC];
        bool pos[VEC];
#pragma unroll
        for (int l = 0; l < VEC; ++l) {
            const Courant c = make_courant(pencil_courant<KIND>(p, o, e0 + l));
            sf[l] = c.sf;
            pos[l] = __double2hiint(c.sf) >= 0;
            cx[l] = pos[l] ? c.c1 : -c.c2;
            cy[l] = pos[l] ? -c.c2 : c.c1;
        }

        // ---- all loads the prologue needs, issued together
        const int M = n - 2;                         // steps whose newest stencil value is an interior load
        const int R = M % (2 * U);                   // peeled in front of the main loop
        T G0 = ldv<VEC>(base), G1 = ldv<VEC>(base + stride);
        T gm2, gm1;
        if (BC == BC_PER) {
            gm2 = ldv<VEC>(base + (long long)(n - 2) * stride);
            gm1 = ldv<VEC>(base + (long long)(n - 1) * stride);
        }
        T hn0, hn1;                                  // BC_HALO: ghost layers above the block
        if (BC == BC_HALO) {
            if (p.halo_lo) {
                const double *h = p.halo_lo + (o * 2) * stride + e0;
                gm2 = ldv<VEC>(h); gm1 = ldv<VEC>(h + stride);
            }
            if (p.halo_hi) {
                const double *h = p.halo_hi + (o * 2) * stride + e0;
                hn0 = ldv<VEC>(h); hn1 = ldv<VEC>(h + stride);
            }
        }
        T pre[2 * U - 1];
#pragma unroll
        for (int u = 0; u < 2 * U - 1; ++u)
            if (u < R) pre[u] = ldv<VEC>(base + (long long)(2 + u) * stride);
        T bufA[U], bufB[U];
        const double *nextp = base + (long long)(2 + R) * stride;       // g_{i+2} of the first main step
        if (R < M) {
#pragma unroll
            for (int u = 0; u < U; ++u) bufA[u] = ldv<VEC>(nextp + (long long)u * stride);
        }
        const T F0 = G0, F1 = G1;                    // originals of cells 0, 1 (periodic wrap)
        if (BC == BC_OUT || (BC == BC_HALO && !p.halo_lo)) { gm2 = G0; gm1 = G0; }
        if (BC == BC_WALL) {
#pragma unroll
            for (int l = 0; l < VEC; ++l) { gm2.v[l] = 0.0; gm1.v[l] = 0.0; }
        }

        double Q[VEC], E[VEC];                       // Q_i, E_i = Q_{i-1} - Q_i
#pragma unroll
        for (int l = 0; l < VEC; ++l) {
            double qm1 = march_q(gm2.v[l], gm1.v[l], G0.v[l], cx[l], cy[l]);
            double q0 = march_q(gm1.v[l], G0.v[l], G1.v[l], cx[l], cy[l]);
            if (BC == BC_WALL) {                     // closed box (R7): face -1/2 carries no flux
                if (pos[l]) qm1 = 0.0; else q0 = 0.0;
            }
            Q[l] = q0;
            E[l] = qm1 - q0;
        }
        double s0[VEC], s1[VEC], s2[VEC];            // sum f, sum vz f, sum vz^2 f along the march (MOM)
#pragma unroll
        for (int l = 0; l < VEC; ++l) { s0[l] = 0.0; s1[l] = 0.0; s2[l] = 0.0; }

        // One march step: nw = g_{i+2} arrives, Q_{i+1} and E_{i+1} are formed, cell i is finished.
        // MODE 0: interior; 1: Q_{i+1} is the cell in front of the high wall (i = n-2);
        // 2: Q_{i+1} is the ghost cell behind it (i = n-1).
        auto step = [&](auto mode_tag, double *dst, const T &nw, double vz) {
            constexpr int MODE = decltype(mode_tag)::value;
            T out;
#pragma unroll
            for (int l = 0; l < VEC; ++l) {
                double qn = march_q(G0.v[l], G1.v[l], nw.v[l], cx[l], cy[l]);
                if (BC == BC_WALL && MODE == 1 && pos[l]) qn = 0.0;      // face n-1/2 carries no flux
                if (BC == BC_WALL && MODE == 2 && !pos[l]) qn = 0.0;
                const double en = Q[l] - qn;
                out.v[l] = fma(sf[l], pos[l] ? E[l] : en, G0.v[l]);
                Q[l] = qn; E[l] = en;
                G0.v[l] = G1.v[l]; G1.v[l] = nw.v[l];
                if (MOM) {
                    const double t = vz * out.v[l];
                    s0[l] += out.v[l]; s1[l] += t; s2[l] = fma(vz, t, s2[l]);
                }
            }
            stv<VEC>(dst, out);
        };
        struct M0 { enum { value = 0 }; }; struct M1 { enum { value = 1 }; }; struct M2 { enum { value = 2 }; };

        double *dst = base;
        const double dvz = p.g.dv[2];
        double vz = MOM ? vcentre(p.g, 2, 0) : 0.0;
        // ---- peeled steps 0 .. R-1
#pragma unroll
        for (int u = 0; u < 2 * U - 1; ++u) {
            if (u < R) {
                step(M0(), dst, pre[u], vz);
                dst += stride;
                if (MOM) vz += dvz;
            }
        }
        // ---- main loop: (M - R) / 2U pairs of chunks, no bounds checks
        const int pairs = (M - R) / (2 * U);
        for (int c = 0; c < pairs; ++c) {
            nextp += (long long)U * stride;
#pragma unroll
            for (int u = 0; u < U; ++u) bufB[u] = ldv<VEC>(nextp + (long long)u * stride);
#pragma unroll
            for (int u = 0; u < U; ++u) {
                step(M0(), dst, bufA[u], vz);
                dst += stride;
                if (MOM) vz += dvz;
            }
            nextp += (long long)U * stride;
            if (c + 1 < pairs) {
#pragma unroll
                for (int u = 0; u < U; ++u) bufA[u] = ldv<VEC>(nextp + (long long)u * stride);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                step(M0(), dst, bufB[u], vz);
                dst += stride;
                if (MOM) vz += dvz;
            }
        }
        // ---- the two steps whose newest stencil value is a ghost cell
        T gn0, gn1;                                  // g_n, g_{n+1}
        if (BC == BC_PER) { gn0 = F0; gn1 = F1; }
        else if (BC == BC_OUT) { gn0 = G1; gn1 = G1; }                  // G1 = g_{n-1} here
        else if (BC == BC_HALO) {
            if (p.halo_hi) { gn0 = hn0; gn1 = hn1; } else { gn0 = G1; gn1 = G1; }
        } else {
#pragma unroll
            for (int l = 0; l < VEC; ++l) { gn0.v[l] = 0.0; gn1.v[l] = 0.0; }
        }
        step(M1(), dst, gn0, vz);
        dst += stride;
        if (MOM) vz += dvz;
        step(M2(), dst, gn1, vz);

        if (MOM) {
            // thread's pencils sit at (jy, jx) = divmod(e0 + l, nvx): combine with vx, vy
#pragma unroll
            for (int l = 0; l < VEC; ++l) {
                const long long e = e0 + l;
                const int jy = (int)(e / p.g.nv[0]), jx = (int)(e - (long long)jy * p.g.nv[0]);
                const double vx = vcentre(p.g, 0, jx), vy = vcentre(p.g, 1, jy);
                const double x0 = vx * s0[l], y0 = vy * s0[l];
                mom[0] += s0[l];
                mom[1] += x0; mom[2] += y0; mom[3] += s1[l];
                mom[4] = fma(vx, x0, mom[4]); mom[5] = fma(vx, y0, mom[5]); mom[6] = fma(vx, s1[l], mom[6]);
                mom[7] = fma(vy, y0, mom[7]); mom[8] = fma(vy, s1[l], mom[8]); mom[9] += s2[l];
            }
        }
    }   // active
    if (MOM) {
        block_reduce_sum<10>(mom, red);
        if (threadIdx.x == 0) {
#pragma unroll
            for (int k = 0; k < 10; ++k) p.mom[(long long)blockIdx.x * 10 + k] = mom[k];
        }
    }
}

// ---------------------------------------------------------------- halo pack
// Copies the two boundary layers of f at one end of a spatial axis (f viewed as [outer][n][inner])
// into buf [outer][2][inner], layers in ascending index order: row0 = 0 (low end) or n-2 (high end).
// 16-byte vector copies when inner is even.
template <int VEC>
__global__ void __launch_bounds__(256)
pack_halo_kernel(const double *__restrict__ f, double *__restrict__ buf, long long outer, int n,
                 long long inner, int row0)
{
    const long long innerV = inner / VEC;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= outer * 2 * innerV) return;
    const long long ol = t / innerV;                 // (o, layer)
    const long long ev = t - ol * innerV;
    const long long o = ol >> 1;
    const int layer = (int)(ol & 1);
    stv<VEC>(buf + ol * inner + ev * VEC, ldv<VEC>(f + (o * n + row0 + layer) * inner + ev * VEC));
}

}  // namespace mphv
