// mphv_kernels.cuh -- hand-written CUDA kernels (sm_100a) of the mphv hot path.
//
// Everything here follows the paper's statement of the method (eq. (1),
// L57 moments, L135 scheme) through the readings R1..R14 of DESIGN.md. It shares no code
// with oracle/ (the CPU test oracle) and includes nothing from it.
//
// Kernel families
//   march_kernel     1-D PFC-3 remap along a STRIDED axis (x, y, z, vy, vz). One thread owns
//                    VEC adjacent pencils (adjacent in the contiguous index), marches along
//                    the axis with a register window and a U-deep register prefetch, in
//                    place. A warp touches 32*VEC*8 contiguous bytes per march step, so
//                    stride-N directions stay coalesced without a transpose.
//   vx_kernel        remap along the CONTIGUOUS axis vx: one thread owns CH consecutive cells
//                    of a row, reads its 2+2 halo through L1, all loads -> barrier -> stores.
//   moments_kernel   one CTA per spatial cell: separable accumulation along vz, then
//                    warp-shuffle + shared-memory block reduction of the 10 moments.
//   shift_kernel     slow path for |s| >= 1 on a periodic axis (whole-cell shift + fractional
//                    remap, out of place through the scratch buffer).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mphv {

enum { BC_PER = 0, BC_OUT = 1, BC_WALL = 2 };
enum { KIND_SPACE = 0, KIND_VEL = 1 };

struct GridDev {
    int nx[3], nv[3];
    double vlo[3], dv[3];   // inactive velocity dim: vlo = -0.5, dv = 1 => centre == 0 exactly
    double qm;
    long long ns;           // spatial cells
    long long nvel;         // velocity cells per spatial cell
};

struct MarchArgs {
    double *f;              // in place
    long long outer;        // f viewed as [outer][n][inner]
    long long inner;        // doubles
    int n;
    int dim;                // swept dimension (spatial 0..2 or velocity 1..2)
    double dt;
    double dx;              // width of the swept cell (dx_d or dv_d)
    const double *E, *B;    // velocity sweeps only
    double *mom;            // fused moments output workspace [10][ns] (vz sweep only) or null
    double dV;
    GridDev g;
};

// ---------------------------------------------------------------- small vector helpers
template <int VEC> struct V { double v[VEC]; };

template <int VEC> __device__ __forceinline__ V<VEC> ldv(const double *p);
template <> __device__ __forceinline__ V<1> ldv<1>(const double *p) { V<1> r; r.v[0] = *p; return r; }
template <> __device__ __forceinline__ V<2> ldv<2>(const double *p)
{
    double2 t = *reinterpret_cast<const double2 *>(p);
    V<2> r; r.v[0] = t.x; r.v[1] = t.y; return r;
}
template <int VEC> __device__ __forceinline__ void stv(double *p, const V<VEC> &x);
template <> __device__ __forceinline__ void stv<1>(double *p, const V<1> &x) { *p = x.v[0]; }
template <> __device__ __forceinline__ void stv<2>(double *p, const V<2> &x)
{
    *reinterpret_cast<double2 *>(p) = make_double2(x.v[0], x.v[1]);
}

// ---------------------------------------------------------------- the scheme (R2, R3)
// Fractional flux through one face, for the upwind triple (a, b, c): b is the cell the
// mass leaves, a the cell behind it, c the cell it enters. sf = signed fractional Courant
// number (+alpha or -beta), c1 = (1-|sf|)(2-|sf|)/6, c2 = (1-|sf|)(1+|sf|)/6.
// Limited slopes are the PFC positivity correctors in division-free form:
//   L+ = d+ > 0 ? min(d+, 2b) : d+,   L- = d- < 0 ? max(d-, -2b) : d-.
// For sf < 0 the caller passes the mirrored triple; the mirror image of the formula is the
// formula of the mirror image (R11), so one expression serves both signs.
__device__ __forceinline__ double face_flux(double a, double b, double c, double sf, double c1, double c2)
{
    const double dp = c - b;
    const double dm = b - a;
    const double cap = b + b;
    const double lp = dp > 0.0 ? fmin(dp, cap) : dp;
    const double lm = dm < 0.0 ? fmax(dm, -cap) : dm;
    return sf * ((b + c1 * lp) + c2 * lm);
}

struct Courant { double sf, c1, c2; bool pos; };

__device__ __forceinline__ Courant make_courant(double s_frac)
{
    Courant c;
    const double fr = fabs(s_frac);
    c.sf = s_frac;
    c.c1 = ((1.0 - fr) * (2.0 - fr)) / 6.0;
    c.c2 = ((1.0 - fr) * (1.0 + fr)) / 6.0;
    c.pos = s_frac >= 0.0;
    return c;
}

// velocity cell centre, evaluated exactly as the paper-level definition x_j = lo + (j+1/2) d
__device__ __forceinline__ double vcentre(const GridDev &g, int d, int j)
{
    return __dadd_rn(g.vlo[d], __dmul_rn((double)j + 0.5, g.dv[d]));
}

// Lorentz acceleration component d (eq. (1)): a_d = (q/m)(E_d + v_a B_b - v_b B_a) with
// a = (d+1)%3, b = (d+2)%3, evaluated product, product, difference, sum, scale (no FMA).
__device__ __forceinline__ double accel(double qm, double Ed, double Ba, double Bb, double va, double vb)
{
    const double cross = __dsub_rn(__dmul_rn(va, Bb), __dmul_rn(vb, Ba));
    return __dmul_rn(qm, __dadd_rn(Ed, cross));
}
__device__ __forceinline__ double accel_at(const GridDev &g, const double *E, const double *B, int d,
                                           long long cell, double va, double vb)
{
    const int ia = (d + 1) % 3, ib = (d + 2) % 3;
    return accel(g.qm, E[d * g.ns + cell], B[ia * g.ns + cell], B[ib * g.ns + cell], va, vb);
}

// Courant number of the pencil through contiguous element e of outer block o.
template <int KIND>
__device__ __forceinline__ double pencil_courant(const MarchArgs &p, long long o, long long e)
{
    const GridDev &g = p.g;
    if (KIND == KIND_SPACE) {
        const long long jv = e % g.nvel;
        int jd;
        if (p.dim == 0)      jd = (int)(jv % g.nv[0]);
        else if (p.dim == 1) jd = (int)((jv / g.nv[0]) % g.nv[1]);
        else                 jd = (int)(jv / ((long long)g.nv[0] * g.nv[1]));
        const double v = vcentre(g, p.dim, jd);
        return __ddiv_rn(__dmul_rn(v, p.dt), p.dx);
    } else {
        long long cell; double va, vb;
        if (p.dim == 2) {                       // vz: outer = cell, inner = (jy, jx); a_z needs (vx, vy)
            cell = o;
            const int jx = (int)(e % g.nv[0]), jy = (int)(e / g.nv[0]);
            va = vcentre(g, 0, jx); vb = vcentre(g, 1, jy);
        } else {                                // vy: outer = (cell, jz), inner = jx; a_y needs (vz, vx)
            cell = o / g.nv[2];
            const int jz = (int)(o % g.nv[2]);
            va = vcentre(g, 2, jz); vb = vcentre(g, 0, (int)e);
        }
        const double a = accel_at(g, p.E, p.B, p.dim, cell, va, vb);
        return __ddiv_rn(__dmul_rn(a, p.dt), p.dx);
    }
}

// ---------------------------------------------------------------- march kernel
// In-place remap with |s| < 1 (k = 0). Window (g_{i-1}, g_i, g_{i+1}, g_{i+2}) in registers;
// buf/nxt hold the next 2U loads so that U independent loads per thread are always in flight.
template <int VEC, int U, int KIND, int BC>
__global__ void __launch_bounds__(256)
march_kernel(const MarchArgs p)
{
    typedef V<VEC> T;
    const long long innerV = p.inner / VEC;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= p.outer * innerV) return;
    const long long o = t / innerV;
    const long long e0 = (t - o * innerV) * VEC;
    const int n = p.n;
    const long long stride = p.inner;
    double *base = p.f + (o * n) * stride + e0;

    Courant cn[VEC];
#pragma unroll
    for (int l = 0; l < VEC; ++l) cn[l] = make_courant(pencil_courant<KIND>(p, o, e0 + l));

    T f0s, f1s;                                  // originals of cells 0, 1 (periodic wrap)
    T gm2, gm1, c0, c1v;
    c0 = ldv<VEC>(base);
    c1v = ldv<VEC>(base + stride);
    f0s = c0; f1s = c1v;
    if (BC == BC_PER) {
        gm2 = ldv<VEC>(base + (long long)(n - 2) * stride);
        gm1 = ldv<VEC>(base + (long long)(n - 1) * stride);
    } else if (BC == BC_OUT) {
        gm2 = c0; gm1 = c0;
    } else {
#pragma unroll
        for (int l = 0; l < VEC; ++l) { gm2.v[l] = 0.0; gm1.v[l] = 0.0; }
    }

    auto fetch = [&](int i) -> T {
        if (i < n) return ldv<VEC>(base + (long long)i * stride);
        if (BC == BC_PER) return (i == n) ? f0s : f1s;
        if (BC == BC_OUT) return ldv<VEC>(base + (long long)(n - 1) * stride);
        T z;
#pragma unroll
        for (int l = 0; l < VEC; ++l) z.v[l] = 0.0;
        return z;
    };

    T buf[U], nxt[U];
#pragma unroll
    for (int u = 0; u < U; ++u) buf[u] = fetch(2 + u);

    // flux through the low face -1/2 (zero for the closed velocity box, R7)
    T phiprev;
#pragma unroll
    for (int l = 0; l < VEC; ++l) {
        if (BC == BC_WALL) phiprev.v[l] = 0.0;
        else {
            const bool ps = cn[l].pos;
            phiprev.v[l] = face_flux(ps ? gm2.v[l] : c1v.v[l], ps ? gm1.v[l] : c0.v[l],
                                     ps ? c0.v[l] : gm1.v[l], cn[l].sf, cn[l].c1, cn[l].c2);
        }
    }
    T a1 = gm1;                                  // g_{i-1}

    for (int i0 = 0; i0 < n; i0 += U) {
#pragma unroll
        for (int u = 0; u < U; ++u) nxt[u] = fetch(i0 + 2 + U + u);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = i0 + u;
            if (i < n) {
                const T c2v = buf[u];            // g_{i+2}
                T out;
#pragma unroll
                for (int l = 0; l < VEC; ++l) {
                    const bool ps = cn[l].pos;
                    double phi = face_flux(ps ? a1.v[l] : c2v.v[l], ps ? c0.v[l] : c1v.v[l],
                                           ps ? c1v.v[l] : c0.v[l], cn[l].sf, cn[l].c1, cn[l].c2);
                    if (BC == BC_WALL && i == n - 1) phi = 0.0;
                    out.v[l] = c0.v[l] + (phiprev.v[l] - phi);
                    phiprev.v[l] = phi;
                }
                stv<VEC>(base + (long long)i * stride, out);
                a1 = c0; c0 = c1v; c1v = c2v;
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) buf[u] = nxt[u];
    }
}

// ---------------------------------------------------------------- vx kernel (contiguous axis)
struct VxArgs {
    double *f;
    long long rows;         // ns * nvz * nvy
    int nvx;
    int rows_per_cta;
    double dt;
    const double *E, *B;
    GridDev g;
};

template <int CH>
__global__ void __launch_bounds__(256)
vx_kernel(const VxArgs p)
{
    const int cpr = p.nvx / CH;                  // chunks per row
    const int rl = threadIdx.x / cpr;
    const int q = threadIdx.x - rl * cpr;
    const long long row = (long long)blockIdx.x * p.rows_per_cta + rl;
    const bool active = rl < p.rows_per_cta && row < p.rows;

    double w[CH + 4];                            // g_{c0-2} .. g_{c0+CH+1}
    Courant cn;
    double *ptr = nullptr;
    if (active) {
        const GridDev &g = p.g;
        ptr = p.f + row * p.nvx + (long long)q * CH;
        if (CH == 1) {
            w[2] = ptr[0];
            w[0] = q >= 2 ? ptr[-2] : 0.0;
            w[1] = q >= 1 ? ptr[-1] : 0.0;
            w[3] = q + 1 < cpr ? ptr[1] : 0.0;
            w[4] = q + 2 < cpr ? ptr[2] : 0.0;
        } else {
#pragma unroll
            for (int c = 0; c < CH; c += 2) {
                const double2 t = *reinterpret_cast<const double2 *>(ptr + c);
                w[2 + c] = t.x; w[3 + c] = t.y;
            }
            if (q > 0) { const double2 t = *reinterpret_cast<const double2 *>(ptr - 2); w[0] = t.x; w[1] = t.y; }
            else { w[0] = 0.0; w[1] = 0.0; }
            if (q + 1 < cpr) { const double2 t = *reinterpret_cast<const double2 *>(ptr + CH); w[CH + 2] = t.x; w[CH + 3] = t.y; }
            else { w[CH + 2] = 0.0; w[CH + 3] = 0.0; }
        }
        // a_x = (q/m)(E_x + vy B_z - vz B_y); row = (cell, jz, jy)
        const long long plane = row / g.nv[1];
        const int jy = (int)(row - plane * g.nv[1]);
        const long long cell = plane / g.nv[2];
        const int jz = (int)(plane - cell * g.nv[2]);
        const double a = accel_at(g, p.E, p.B, 0, cell, vcentre(g, 1, jy), vcentre(g, 2, jz));
        cn = make_courant(__ddiv_rn(__dmul_rn(a, p.dt), g.dv[0]));
    }
    __syncthreads();                             // every load of the CTA precedes every store
    if (!active) return;

    // faces c0-1/2 .. c0+CH-1/2; face m lies between w[m+1] and w[m+2]
    double phi[CH + 1];
#pragma unroll
    for (int m = 0; m <= CH; ++m) {
        const bool ps = cn.pos;
        phi[m] = face_flux(ps ? w[m] : w[m + 3], ps ? w[m + 1] : w[m + 2], ps ? w[m + 2] : w[m + 1],
                           cn.sf, cn.c1, cn.c2);
    }
    if (q == 0) phi[0] = 0.0;                    // closed velocity box (R7)
    if (q == cpr - 1) phi[CH] = 0.0;
    if (CH == 1) {
        ptr[0] = w[2] + (phi[0] - phi[1]);
    } else {
#pragma unroll
        for (int c = 0; c < CH; c += 2) {
            const double o0 = w[2 + c] + (phi[c] - phi[c + 1]);
            const double o1 = w[3 + c] + (phi[c + 1] - phi[c + 2]);
            *reinterpret_cast<double2 *>(ptr + c) = make_double2(o0, o1);
        }
    }
}

// ---------------------------------------------------------------- shift kernel (slow path)
// Periodic axis, any s: g_i = f_{i-k}, k = trunc(s), then the fractional remap with
// sf = s - k. Out of place (src -> dst), one thread per pencil, modular indexing.
__global__ void __launch_bounds__(256)
shift_kernel(const MarchArgs p, const double *__restrict__ src, double *__restrict__ dst)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= p.outer * p.inner) return;
    const long long o = t / p.inner;
    const long long e = t - o * p.inner;
    const int n = p.n;
    const long long stride = p.inner;
    const double *sb = src + (o * n) * stride + e;
    double *db = dst + (o * n) * stride + e;
    const double s = pencil_courant<KIND_SPACE>(p, o, e);
    const double kf = trunc(s);
    const Courant cn = make_courant(s - kf);
    long long km = (long long)fmod(kf, (double)n);      // |km| < n
    auto g = [&](int i) -> double {
        long long m = ((long long)i - km) % n;
        if (m < 0) m += n;
        return sb[m * stride];
    };
    auto flux = [&](int i) -> double {                  // face i+1/2
        return cn.pos ? face_flux(g(i - 1), g(i), g(i + 1), cn.sf, cn.c1, cn.c2)
                      : face_flux(g(i + 2), g(i + 1), g(i), cn.sf, cn.c1, cn.c2);
    };
    double phiprev = flux(-1);
    for (int i = 0; i < n; ++i) {
        const double phi = flux(i);
        db[(long long)i * stride] = g(i) + (phiprev - phi);
        phiprev = phi;
    }
}

// ---------------------------------------------------------------- block reduction helper
template <int NV>
__device__ __forceinline__ void block_reduce_sum(double (&val)[NV], double *smem /* [NV][32] */)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double x = val[k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
        if (lane == 0) smem[k * 32 + wid] = x;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double x = lane < nw ? smem[k * 32 + lane] : 0.0;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
            val[k] = x;
        }
    }
}

// ---------------------------------------------------------------- moments kernel
// One CTA per spatial cell. Thread <-> (jy, jx) position(s); marches over jz accumulating
// S0 = sum f, S1 = sum vz f, S2 = sum vz^2 f (3 FMA per cell), then combines with vx, vy.
struct MomArgs {
    const double *f;
    double *n, *j, *P;
    double dV;
    GridDev g;
};

__global__ void __launch_bounds__(512)
moments_kernel(const MomArgs p)
{
    __shared__ double red[10 * 32];
    const GridDev &g = p.g;
    const long long cell = blockIdx.x;
    const double *cube = p.f + cell * g.nvel;
    const int plane = g.nv[0] * g.nv[1];
    double m[10];
#pragma unroll
    for (int k = 0; k < 10; ++k) m[k] = 0.0;
    for (int pos = threadIdx.x; pos < plane; pos += blockDim.x) {
        const int jy = pos / g.nv[0], jx = pos - jy * g.nv[0];
        const double vx = vcentre(g, 0, jx), vy = vcentre(g, 1, jy);
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;
        for (int jz = 0; jz < g.nv[2]; ++jz) {
            const double fv = cube[(long long)jz * plane + pos];
            const double vz = vcentre(g, 2, jz);
            const double t = vz * fv;
            s0 += fv; s1 += t; s2 = fma(vz, t, s2);
        }
        const double x0 = vx * s0, y0 = vy * s0;
        m[0] += s0;
        m[1] += x0; m[2] += y0; m[3] += s1;
        m[4] = fma(vx, x0, m[4]); m[5] = fma(vx, y0, m[5]); m[6] = fma(vx, s1, m[6]);
        m[7] = fma(vy, y0, m[7]); m[8] = fma(vy, s1, m[8]); m[9] += s2;
    }
    block_reduce_sum<10>(m, red);
    if (threadIdx.x == 0) {
        p.n[cell] = m[0] * p.dV;
#pragma unroll
        for (int a = 0; a < 3; ++a) p.j[a * g.ns + cell] = m[1 + a] * p.dV;
#pragma unroll
        for (int a = 0; a < 6; ++a) p.P[a * g.ns + cell] = m[4 + a] * p.dV;
    }
}

// ---------------------------------------------------------------- sum of f (mass)
// Stage 1: grid-stride, Kahan-compensated per thread, block tree -> partial[blockIdx.x].
// Stage 2 (one block): same over the partials. Fixed order => deterministic.
__global__ void __launch_bounds__(256)
sum_kernel(const double *__restrict__ x, long long count, double *__restrict__ partial)
{
    __shared__ double red[32];
    double s = 0.0, c = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < count;
         i += (long long)gridDim.x * blockDim.x) {
        const double y = x[i] - c;
        const double tt = s + y;
        c = (tt - s) - y;
        s = tt;
    }
    double v[1] = { s };
    block_reduce_sum<1>(v, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = v[0];
}

// ---------------------------------------------------------------- max |a_d| over cells
// The acceleration is linear in the two other velocity components, and fp64 rounding is
// monotone, so its extreme over the velocity grid is at one of the four corner centres.
__global__ void __launch_bounds__(1024)
amax_kernel(const double *__restrict__ E, const double *__restrict__ B, GridDev g, double *out /* [3] */)
{
    __shared__ double red[3][32];
    double mx[3] = { 0.0, 0.0, 0.0 };
    bool bad[3] = { false, false, false };
    for (long long cell = threadIdx.x; cell < g.ns; cell += blockDim.x) {
        for (int d = 0; d < 3; ++d) {
            const int da = (d + 1) % 3, db = (d + 2) % 3;
            for (int ca = 0; ca < 2; ++ca)
                for (int cb = 0; cb < 2; ++cb) {
                    const double va = vcentre(g, da, ca ? g.nv[da] - 1 : 0);
                    const double vb = vcentre(g, db, cb ? g.nv[db] - 1 : 0);
                    const double a = fabs(accel_at(g, E, B, d, cell, va, vb));
                    if (!(a == a)) bad[d] = true;
                    mx[d] = fmax(mx[d], a);
                }
        }
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int d = 0; d < 3; ++d) {
        double x = bad[d] ? __longlong_as_double(0x7ff8000000000000LL) : mx[d];
        for (int off = 16; off > 0; off >>= 1) {
            const double y = __shfl_down_sync(0xffffffffu, x, off);
            x = (x != x || y != y) ? __longlong_as_double(0x7ff8000000000000LL) : fmax(x, y);
        }
        if (lane == 0) red[d][wid] = x;
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        const int d = threadIdx.x;
        double x = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
            const double y = red[d][w];
            x = (x != x || y != y) ? __longlong_as_double(0x7ff8000000000000LL) : fmax(x, y);
        }
        out[d] = x;
    }
}

}  // namespace mphv
