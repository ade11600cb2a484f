// mphv_sxy.cuh -- the spatial sweeps S_x and S_y (free streaming v . grad_x f of eq. (1), P:L53;
// scheme P:L135, readings R2/R3/R6/R11; order x then y, R5) in ONE pass over f.
//
// f is [outer = nz][ny][nx][nvel] with the velocity index contiguous. A CTA owns a chunk of C
// consecutive velocity indices (C * 8 = 128 or 64 bytes) of one z slab, for ALL x and y, and
// marches along y:
//
//   row stream   the raw row y (nx pieces of C doubles, strided by nvel) is brought into an NR-deep
//                shared-memory ring with 16-byte cp.async copies, NR-1 rows ahead of its use --
//                no registers are tied up by loads in flight;
//   S_x          thread <-> (4 consecutive x cells, one velocity index): 7 values of the row from
//                shared memory (the window starts one cell later for s < 0, so lanes of either sign
//                run the same code), 5 cell fluxes Q, 4 new cells -- they stay in REGISTERS;
//   S_y          those 4 cells are the newest entries of four register windows marching along y
//                (the row stream IS the y march; cell-based form of mphv_march.cuh): the finished
//                row y-2 is stored straight to global memory, in place (its raw data were consumed
//                two rows ago; a CTA never touches another CTA's chunk).
//
// Periodic y: the rows ny-2, ny-1 are produced first (and again at the end of the stream, before
// they are overwritten), the S_x images of rows 0, 1 are kept for the wrap. Outflow: zero-gradient
// ghosts (R6). Boundary handling in x is index math on the 7 shared-memory offsets of a thread.
// BCX = BC_HALO: the block is one of several along x; the ghost cells of every row come from the
// neighbours' packed boundary layers. Requires nx % 4 == 0, nvel % C == 0, |s| < 1 on both axes; other
// cases use the march kernels.
#pragma once
#include "mphv_vstage.cuh"

namespace mphv {

struct SxyArgs {
    double *f;
    int nx, ny;
    int chunks;             // nvel / C
    long long nvel;         // doubles between x neighbours
    double dt, dx, dy;
    // BCX == BC_HALO (block decomposition along x): the two ghost layers below / above the block,
    // each [nz ny][2][nvel] as packed by pack_halo_kernel; NULL = global outflow end (zero-gradient ghosts, R6)
    const double *halo_lo, *halo_hi;
    GridDev g;
};

__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src_gmem)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// ring-row offset (doubles) of cell x: C doubles per cell; with C = 8 a pad of 8 doubles after every
// 4 cells, so that the two x groups of a half-warp hit different banks
template <int C> __device__ __forceinline__ int sxy_xoff(int x)
{
    return C == 8 ? x * 8 + (x >> 2) * 8 : x * C;
}
template <int C> __host__ __device__ inline int sxy_row_doubles(int nx)
{
    return C == 8 ? nx * 8 + (nx / 4) * 8 : nx * C;
}

template <int C, int NR, int BCX, int BCY, int TMAX, int MINB>
__global__ void __launch_bounds__(TMAX, MINB)
sxy_kernel(const SxyArgs p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);                 // [NR][rowd]
    const int nx = p.nx, ny = p.ny;
    constexpr int XS = BCX == BC_HALO ? 2 : 0;                           // ring rows carry 2 + 2 ghost cells
    const int rowd = sxy_row_doubles<C>(nx + 2 * XS);
    const int tid = threadIdx.x, T = blockDim.x;                         // T = (nx / 4) * C
    double *keep = ring + (size_t)NR * rowd;                             // [2][4][T] (periodic y only)
    const int v = tid % C, xq = tid / C;
    const int x0 = 4 * xq;
    const long long o = blockIdx.x / p.chunks;
    const int chunk = (int)(blockIdx.x - o * p.chunks);
    const long long nvel = p.nvel;
    const long long row_stride = (long long)nx * nvel;
    double *slab = p.f + o * ny * row_stride + (long long)chunk * C;     // cell (y, x): slab + y row_stride + x nvel

    // ---- Courant data of the thread's velocity index: s_x from jvx, s_y from jvy
    const long long jv = (long long)chunk * C + v;
    const int jvx = (int)(jv % p.g.nv[0]);
    const int jvy = (int)((jv / p.g.nv[0]) % p.g.nv[1]);
    const double sx = __ddiv_rn(__dmul_rn(vcentre(p.g, 0, jvx), p.dt), p.dx);
    const double sy = __ddiv_rn(__dmul_rn(vcentre(p.g, 1, jvy), p.dt), p.dy);
    double c1, nc2;
    courant_poly(sx, c1, nc2);
    const bool posx = __double2hiint(sx) >= 0;
    const double xcx = posx ? c1 : nc2, xcy = posx ? nc2 : c1;
    courant_poly(sy, c1, nc2);
    const bool posy = __double2hiint(sy) >= 0;
    const double ycx = posy ? c1 : nc2, ycy = posy ? nc2 : c1;

    // ---- the 7 cells of the S_x window: x0-2 .. x0+4 (s >= 0) or x0-1 .. x0+5 (s < 0)
    int off[7];
#pragma unroll
    for (int m = 0; m < 7; ++m) {
        int xi = x0 - 2 + (posx ? 0 : 1) + m;
        if (BCX == BC_PER) { if (xi < 0) xi += nx; else if (xi >= nx) xi -= nx; }
        else if (BCX == BC_OUT) { xi = xi < 0 ? 0 : (xi >= nx ? nx - 1 : xi); }
        else {
            if (xi < 0 && !p.halo_lo) xi = 0;
            if (xi >= nx && !p.halo_hi) xi = nx - 1;
        }
        off[m] = sxy_xoff<C>(xi + XS) + v;
    }

    // ---- row stream: production k brings row row_of(k); K productions
    const int K = BCY == BC_PER ? ny + 2 : ny;
    auto row_of = [&](int k) { return BCY == BC_PER ? (k < 2 ? ny - 2 + k : k - 2) : k; };
    auto issue_row = [&](int k) {
        double *dst = ring + (size_t)(k % NR) * rowd;
        const double *src = slab + (long long)row_of(k) * row_stride;
#pragma unroll
        for (int u = 0; u < 2; ++u) {                                    // nx C / 2 pieces of 16 bytes = 2 T
            const int piece = tid + u * T;
            const int x = piece / (C / 2), part = piece % (C / 2);
            cp_async16(dst + sxy_xoff<C>(x + XS) + 2 * part, src + (long long)x * nvel + 2 * part);
        }
        if (BCX == BC_HALO && tid < 4 * (C / 2)) {                       // the 2 + 2 ghost cells of the row
            const int hx = tid / (C / 2), part = tid % (C / 2);
            const double *h = hx < 2 ? p.halo_lo : p.halo_hi;
            if (h)
                cp_async16(dst + sxy_xoff<C>(hx < 2 ? hx : nx + hx) + 2 * part,
                           h + ((o * ny + row_of(k)) * 2 + (hx & 1)) * nvel + (long long)chunk * C + 2 * part);
        }
    };
#pragma unroll
    for (int k = 0; k < NR - 1; ++k) {
        if (k < K) issue_row(k);
        cp_async_commit();
    }

    // S_x of the row of production k: the thread's 4 new cells
    auto produce = [&](int k, double (&nw)[4]) {
        cp_async_wait<NR - 2>();                     // this thread's pieces of row k have landed
        __syncthreads();                             // everyone's have; the slot of production k-1 is free
        if (k + NR - 1 < K) issue_row(k + NR - 1);
        cp_async_commit();
        const double *row = ring + (size_t)(k % NR) * rowd;
        double w[7], q[5];
#pragma unroll
        for (int m = 0; m < 7; ++m) w[m] = row[off[m]];
        march_q_window<5>(w, xcx, xcy, q);
#pragma unroll
        for (int c = 0; c < 4; ++c) nw[c] = fma(sx, q[c] - q[c + 1], posx ? w[c + 2] : w[c + 1]);
    };

    double G0[4], G1[4], Q[4], E[4];                 // g_i, g_{i+1}, Q_i, E_i = Q_{i-1} - Q_i along y
    int k = 0;
    {
        double gm2[4], gm1[4];
        if (BCY == BC_PER) { produce(k++, gm2); produce(k++, gm1); }
        produce(k++, G0);
        produce(k++, G1);
        if (BCY == BC_PER) {
#pragma unroll
            for (int m = 0; m < 4; ++m) { keep[m * T + tid] = G0[m]; keep[(4 + m) * T + tid] = G1[m]; }
        } else {
#pragma unroll
            for (int m = 0; m < 4; ++m) { gm2[m] = G0[m]; gm1[m] = G0[m]; }
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double qm1 = march_q(gm2[m], gm1[m], G0[m], ycx, ycy);
            const double q0 = march_q(gm1[m], G0[m], G1[m], ycx, ycy);
            Q[m] = q0; E[m] = qm1 - q0;
        }
    }
    // one y march step: nw = g_{i+2} arrives, Q_{i+1} is formed, row i is finished and stored
    double *dst = slab + (long long)x0 * nvel + v;
    auto ystep = [&](const double (&nw)[4]) {
        double qn[4];
        march_q_lanes<4>(G0, G1, nw, ycx, ycy, qn);
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double en = Q[m] - qn[m];
            const double out = fma(sy, posy ? E[m] : en, G0[m]);
            if (BCX == BC_HALO) dst[m * nvel] = out;     // (measured: the streaming store slows the halo variant)
            else __stcs(dst + m * nvel, out);            // streaming store: f is not re-read before the next kernel
            Q[m] = qn[m]; E[m] = en;
            G0[m] = G1[m]; G1[m] = nw[m];
        }
        dst += row_stride;
    };
#pragma unroll 3
    for (; k < K; ++k) {                             // unrolled by the period of the (G0, G1, nw) rotation
        double nw[4];
        produce(k, nw);
        ystep(nw);
    }
    // the two steps whose newest stencil value is a ghost row
    {
        double gn[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) gn[m] = BCY == BC_PER ? keep[m * T + tid] : G1[m];
        ystep(gn);
#pragma unroll
        for (int m = 0; m < 4; ++m) gn[m] = BCY == BC_PER ? keep[(4 + m) * T + tid] : G1[m];
        ystep(gn);
    }
}

}  // namespace mphv
