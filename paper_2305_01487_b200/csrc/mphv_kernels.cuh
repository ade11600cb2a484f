// mphv_kernels.cuh -- hand-written CUDA kernels (sm_100a) of the mphv hot path.
//
// Everything here follows the paper's statement of the method (eq. (1),
// L57 moments, L135 scheme) through the readings R1..R14 of DESIGN.md. It shares no code
// with oracle/ (the CPU test oracle) and includes nothing from it.
//
// Kernel families
//   march2_kernel    (mphv_march.cuh) 1-D PFC-3 remap along a STRIDED axis (x, y, z, vy, vz),
//                    in place, one thread per VEC adjacent pencils.
//   vcube_kernel     (mphv_vcube.cuh) V_vx + V_vy [+ V_vz + moments] per velocity plane stream.
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

enum { BC_PER = 0, BC_OUT = 1, BC_WALL = 2, BC_HALO = 3 };
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
    double *mom;            // fused moments: per-CTA partials [ns*tiles][10] (vz sweep only) or null
    int tiles, per_tile;    // CTA tiling of the fused-moments variant
    double dV;
    // BC_HALO (spatial block decomposition): the two ghost layers below / above the block,
    // each [outer][2][inner] (layers in ascending index order). NULL = that end is a global outflow
    // end (zero-gradient ghosts, R6).
    const double *halo_lo, *halo_hi;
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
    const double lp = (dp > 0.0 && cap < dp) ? cap : dp;      // d+ > 0 ? min(d+, 2b) : d+
    const double lm = (dm < 0.0 && dm < -cap) ? -cap : dm;    // d- < 0 ? max(d-, -2b) : d-
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

// ---------------------------------------------------------------- march kernel: mphv_march.cuh

// Sums the per-CTA partial moments of the fused V_vz kernel in fixed order and scales by dV.
__global__ void __launch_bounds__(256)
mom_finalize_kernel(const double *__restrict__ part, int tiles, long long ns, double dV,
                    double *__restrict__ n, double *__restrict__ j, double *__restrict__ P)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ns * 10) return;
    const long long cell = t / 10;
    const int k = (int)(t - cell * 10);
    double acc = 0.0;
    for (int tl = 0; tl < tiles; ++tl) acc += part[(cell * tiles + tl) * 10 + k];
    acc *= dV;
    if (k == 0) n[cell] = acc;
    else if (k < 4) j[(k - 1) * ns + cell] = acc;
    else P[(k - 4) * ns + cell] = acc;
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

// ---------------------------------------------------------------- fused V_vx + V_vy plane kernel
// One (spatial cell, jvz) plane of nvy x nvx doubles is contiguous in memory (12.8 KB at 40^2).
// Persistent CTAs loop over planes. A plane is brought into shared memory by ONE bulk async
// copy (cp.async.bulk, TMA engine, completion on an mbarrier), NS planes in flight per CTA, so
// no registers are tied up by loads in flight. The vx remap reads the plane from smem and
// writes the result to a second smem buffer; the vy remap reads that buffer and stores straight
// to global memory (in place: the input plane already sits in smem). f is read once and
// written once for both sweeps.
//   vx items: (row r, column pair q): 3 face fluxes for 2 cells;   smem address = 16 * item
//   vy items: (row pair rp, column pair q): 3 face fluxes x 2 columns for 4 cells
// Courant numbers are per row (vx) / per column (vy); they are computed once per plane into
// smem by the first nvy + nvx threads (double-buffered by plane parity).
struct PlaneArgs {
    double *f;
    long long planes;       // ns * nvz
    int nvx, nvy, nvz;
    int hx, hy;             // nvx / 2, nvy / 2
    float inv_hx;           // 1 / hx for the item -> (row, pair) split
    double dt;
    const double *E, *B;
    GridDev g;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Blocks until the phase with the given parity has completed. The suspend-time hint lets the
// hardware park the warp instead of re-issuing the try_wait (a spinning warp costs issue slots).
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity), "r"(20000u) : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void split_item(int item, int h, float inv_h, int &r, int &q)
{
    r = __float2int_rd(((float)item + 0.5f) * inv_h);
    q = item - r * h;
}

// Courant triple from a signed Courant number, with the polynomial constants by multiplication
__device__ __forceinline__ void courant3(double s, double &sf, double &c1, double &c2)
{
    const double fr = fabs(s);
    const double om = 1.0 - fr;
    sf = s;
    c1 = (om * (2.0 - fr)) * (1.0 / 6.0);
    c2 = (om * (1.0 + fr)) * (1.0 / 6.0);
}

template <int NS>
__global__ void __launch_bounds__(448, 2)
vxy_kernel(const PlaneArgs p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int T = blockDim.x;
    const int tid = threadIdx.x;
    const int nvx = p.nvx, nvy = p.nvy, hx = p.hx, hy = p.hy;
    const int cells = nvx * nvy;
    const uint32_t plane_bytes = (uint32_t)cells * 8u;
    double *inbuf = reinterpret_cast<double *>(smem_raw);                 // [NS][cells]
    double *xbuf = inbuf + (size_t)NS * cells;                           // [cells]
    double *cx = xbuf + cells;                                           // [2][3][nvy]  row Courant triples
    double *cy = cx + 6 * nvy;                                           // [2][3][nvx]  column Courant triples
    uint64_t *bars = reinterpret_cast<uint64_t *>(cy + 6 * nvx);         // [NS]

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(&bars[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const long long first = blockIdx.x;
    const long long step = gridDim.x;
    const long long K = first < p.planes ? (p.planes - first + step - 1) / step : 0;

    if (tid == 0) {
        for (int k = 0; k < NS - 1 && k < K; ++k) {
            mbar_expect_tx(&bars[k], plane_bytes);
            bulk_load(inbuf + (size_t)k * cells, p.f + (first + k * step) * cells, plane_bytes, &bars[k]);
        }
    }

    const double dtdvx = p.dt / p.g.dv[0];
    const double dtdvy = p.dt / p.g.dv[1];

    for (long long k = 0; k < K; ++k) {
        const long long plane = first + k * step;
        const int slot = (int)(k % NS);
        const uint32_t parity = (uint32_t)((k / NS) & 1);
        const int par = (int)(k & 1);
        double *cxp = cx + par * 3 * nvy;
        double *cyp = cy + par * 3 * nvx;

        // prefetch plane k+NS-1 into the slot consumed in iteration k-1 (all threads passed S2 of k-1)
        if (tid == 0 && k + NS - 1 < K) {
            const int ns_slot = (int)((k + NS - 1) % NS);
            mbar_expect_tx(&bars[ns_slot], plane_bytes);
            bulk_load(inbuf + (size_t)ns_slot * cells, p.f + (plane + (NS - 1) * step) * cells, plane_bytes, &bars[ns_slot]);
        }

        // Courant numbers of this plane: rows (a_x needs vy, vz) and columns (a_y needs vz, vx)
        {
            const long long cell = plane / p.nvz;
            const int jz = (int)(plane - cell * p.nvz);
            if (tid < nvy) {
                const double a = accel_at(p.g, p.E, p.B, 0, cell, vcentre(p.g, 1, tid), vcentre(p.g, 2, jz));
                double sf, c1, c2;
                courant3(a * dtdvx, sf, c1, c2);
                cxp[tid] = sf; cxp[nvy + tid] = c1; cxp[2 * nvy + tid] = c2;
            } else if (tid >= T - nvx) {
                const int jx = tid - (T - nvx);
                const double a = accel_at(p.g, p.E, p.B, 1, cell, vcentre(p.g, 2, jz), vcentre(p.g, 0, jx));
                double sf, c1, c2;
                courant3(a * dtdvy, sf, c1, c2);
                cyp[jx] = sf; cyp[nvx + jx] = c1; cyp[2 * nvx + jx] = c2;
            }
        }
        mbar_wait(&bars[slot], parity);
        __syncthreads();                         // S1: Courant numbers visible; xbuf free (vy of k-1 done)

        // ---- vx remap: inbuf[slot] -> xbuf
        const double2 *in2 = reinterpret_cast<const double2 *>(inbuf + (size_t)slot * cells);
        double2 *xb2 = reinterpret_cast<double2 *>(xbuf);
        for (int item = tid; item < nvy * hx; item += T) {
            int r, q;
            split_item(item, hx, p.inv_hx, r, q);
            const double2 own = in2[item];
            double2 lft = make_double2(0.0, 0.0), rgt = make_double2(0.0, 0.0);
            if (q > 0) lft = in2[item - 1];
            if (q < hx - 1) rgt = in2[item + 1];
            const double sf = cxp[r], c1 = cxp[nvy + r], c2 = cxp[2 * nvy + r];
            double ph0, ph1, ph2;
            if (sf >= 0.0) {
                ph0 = face_flux(lft.x, lft.y, own.x, sf, c1, c2);
                ph1 = face_flux(lft.y, own.x, own.y, sf, c1, c2);
                ph2 = face_flux(own.x, own.y, rgt.x, sf, c1, c2);
            } else {
                ph0 = face_flux(own.y, own.x, lft.y, sf, c1, c2);
                ph1 = face_flux(rgt.x, own.y, own.x, sf, c1, c2);
                ph2 = face_flux(rgt.y, rgt.x, own.y, sf, c1, c2);
            }
            if (q == 0) ph0 = 0.0;               // closed velocity box (R7)
            if (q == hx - 1) ph2 = 0.0;
            xb2[item] = make_double2(own.x + (ph0 - ph1), own.y + (ph1 - ph2));
        }
        __syncthreads();                         // S2: xbuf complete; inbuf[slot] free for the next bulk load

        // ---- vy remap: xbuf -> global (rows 2rp, 2rp+1 of column pair q)
        double2 *out2 = reinterpret_cast<double2 *>(p.f + plane * cells);
        for (int item = tid; item < hy * hx; item += T) {
            int rp, q;
            split_item(item, hx, p.inv_hx, rp, q);
            const int r0 = 2 * rp;
            double2 w[6];
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                const int r = r0 - 2 + j;
                w[j] = (r >= 0 && r < nvy) ? xb2[r * hx + q] : make_double2(0.0, 0.0);
            }
            const double2 sf = *reinterpret_cast<const double2 *>(cyp + 2 * q);
            const double2 c1 = *reinterpret_cast<const double2 *>(cyp + nvx + 2 * q);
            const double2 c2 = *reinterpret_cast<const double2 *>(cyp + 2 * nvx + 2 * q);
            double a0, a1, a2, b0, b1, b2;
            if (sf.x >= 0.0) {
                a0 = face_flux(w[0].x, w[1].x, w[2].x, sf.x, c1.x, c2.x);
                a1 = face_flux(w[1].x, w[2].x, w[3].x, sf.x, c1.x, c2.x);
                a2 = face_flux(w[2].x, w[3].x, w[4].x, sf.x, c1.x, c2.x);
            } else {
                a0 = face_flux(w[3].x, w[2].x, w[1].x, sf.x, c1.x, c2.x);
                a1 = face_flux(w[4].x, w[3].x, w[2].x, sf.x, c1.x, c2.x);
                a2 = face_flux(w[5].x, w[4].x, w[3].x, sf.x, c1.x, c2.x);
            }
            if (sf.y >= 0.0) {
                b0 = face_flux(w[0].y, w[1].y, w[2].y, sf.y, c1.y, c2.y);
                b1 = face_flux(w[1].y, w[2].y, w[3].y, sf.y, c1.y, c2.y);
                b2 = face_flux(w[2].y, w[3].y, w[4].y, sf.y, c1.y, c2.y);
            } else {
                b0 = face_flux(w[3].y, w[2].y, w[1].y, sf.y, c1.y, c2.y);
                b1 = face_flux(w[4].y, w[3].y, w[2].y, sf.y, c1.y, c2.y);
                b2 = face_flux(w[5].y, w[4].y, w[3].y, sf.y, c1.y, c2.y);
            }
            if (rp == 0) { a0 = 0.0; b0 = 0.0; }
            if (rp == hy - 1) { a2 = 0.0; b2 = 0.0; }
            out2[r0 * hx + q] = make_double2(w[2].x + (a0 - a1), w[2].y + (b0 - b1));
            out2[(r0 + 1) * hx + q] = make_double2(w[3].x + (a1 - a2), w[3].y + (b1 - b2));
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

// deferred RANGE check of the velocity sweeps (no host round trip): bound[d] = max |a_d| (plain mode, scaled here
// by dt / dv_d as the host check does) or max |s_face| (backsubstitution, scale 1); *flag becomes 1 and stays 1
// when a bound is not below 1.
__global__ void range_flag_kernel(const double *bound, double dt, double dv0, double dv1, double dv2, int active, int scaled, double *flag)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const double dv[3] = { dv0, dv1, dv2 };
    bool bad = false;
    for (int d = 0; d < 3; ++d) {
        if (!((active >> d) & 1)) continue;
        const double s = scaled ? fabs(__ddiv_rn(__dmul_rn(bound[d], dt), dv[d])) : bound[d];
        if (!(s * (1.0 + 1.0e-15) < 1.0)) bad = true;
    }
    if (bad) *flag = 1.0;
}

}  // namespace mphv
