// mphv.cu -- the C-ABI boundary of include/mphv.h: argument validation, range checks,
// launch configuration. All arithmetic of the method runs in the kernels of
// mphv_kernels.cuh; there is no CPU fallback.
#include "../../include/mphv.h"
#include "mphv_kernels.cuh"
#include "mphv_vcube.cuh"
#include "mphv_march.cuh"
#include "mphv_vstage.cuh"
#include "mphv_vstage2.cuh"
#include "mphv_vstage3.cuh"
#include "mphv_sxy.cuh"
#include "mphv_backsub.cuh"
#include "mphv_vstage_bs.cuh"
#include "mphv_vstage3_bs.cuh"
#include "mphv_maxwell.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

using namespace mphv;

// slab pipeline of mphv_run_host (see pipe_step)
struct HostPipe {
    int axis, K;
    std::vector<mphv_ctx *> sub;
    std::vector<int> row0;                    // first index of slab k along axis; row0[K] = n
    double *halo;                             // [K][2 sides][halo_count of the thickest slab]
    double *fld;                              // [K] x ([3][ns_k] E | [3][ns_k] B)
    double *mom;                              // [10][ns_k max]
    size_t halo_stride, layer;                // doubles per (slab, side); cells per index along axis
    cudaStream_t h2d, d2h;
    std::vector<cudaEvent_t> ev_in, ev_out;
};

struct mphv_ctx {
    mphv_grid grid;
    mphv_box box;
    double qm;
    int dev;                 // CUDA device the context was created on (every entry point runs on it)
    cudaStream_t stream;
    double *f, *scratch;
    const double *E, *B;
    size_t ns, nvel, nf;
    double dx[3], dv[3];
    GridDev gd;
    double amax[3];          // max |a_d| over all pencils, from the last set_fields
    bool deferred;           // mphv_set_fields_deferred: the bounds stay on the device, RANGE checks raise a device flag
    double *fld;             // device copy of host fields for mphv_step_fields_host: [3 ns] E | [3 ns] B (lazy)
    double *ws;              // device workspace: [10 ns] moments | [10 ns mom_tiles] partials | [SUM_BLOCKS] | [8]
    int mom_tiles, mom_per_tile, mom_block;   // CTA tiling of the fused V_vz + moments kernel
    int sm_count;
    int vxy_T, vxy_grid; size_t vxy_smem;     // fused V_vx + V_vy plane kernel launch shape (0 = unsupported)
    int vs_T, vs_grid, vs_variant, vs_bs; size_t vs_smem;
    int vs3_T, vs3_grid, vs3_bs; size_t vs3_smem;            // fourth-generation (warp-specialised) whole-V-stage kernel, plain mode (T = 0: shape not covered)
    int vs2_T, vs2_grid; size_t vs2_smem;            // third-generation whole-V-stage kernel, plain mode (T = 0: shape not covered)
    int sxy_T, sxy_C; size_t sxy_smem;               // fused S_x + S_y kernel (T = 0: unsupported)
    int cube_T, cube_grid, cube_variant, plane_grid; size_t cube_smem, plane_smem;  // whole-V-stage cube kernel launch shape (T = 0: unsupported)
    int vmode;                                       // 0 plain V sweeps, 1 backsubstitution
    double *bs_K;                                    // device [ns][12] face-displacement coefficients + [3] maxima
    double bs_dt; bool bs_valid; double bs_smax[3];
    struct HostPipe *pipe;   // slab pipeline of mphv_run_host (lazy)
    bool pipe_failed;        // building it failed once (out of memory): not tried again, mphv_run_host takes the plain path
    uint64_t launches;
    int fusion;
    int vs_gen_max;          // newest generation of the whole-V-stage kernel the launcher may pick (mphv_set_vstage_generation)
    int timing;
    struct Pending { int slot; cudaEvent_t e0, e1; };
    std::vector<Pending> *pending;
    double slot_ms[24];
    uint64_t slot_launches[24];
    double slot_bytes[24];
    double slot_moved[24];
    char err[512];
};

enum { SLOT_SX0 = 0, SLOT_SX1, SLOT_SX2, SLOT_VX, SLOT_VY, SLOT_VZ, SLOT_MOM, SLOT_VXY, SLOT_VZMOM,
       SLOT_SHIFT, SLOT_SUM, SLOT_AMAX, SLOT_VCUBE, SLOT_VCUBE_MOM, SLOT_PACK, SLOT_SXY, SLOT_BSCOEF, SLOT_MAXW, SLOT_EXCH, SLOT_MATCH, SLOT_COUNT };
static const char *const SLOT_NAMES[SLOT_COUNT] = {
    "sweep_x0", "sweep_x1", "sweep_x2", "sweep_vx", "sweep_vy", "sweep_vz", "moments",
    "fused_vx_vy", "fused_vz_moments", "shift_periodic", "sum_f", "amax_fields",
    "fused_vx_vy_vz", "fused_vx_vy_vz_moments", "pack_halo", "fused_sx_sy", "backsub_coefficients", "maxwellian", "exchange_maxwellian", "match_moments" };

namespace {

const int SUM_BLOCKS = 1184;           // 8 x 148 SMs
char g_create_err[512] = "";

void set_err(mphv_ctx *c, const char *fmt, ...)
{
    char *dst = c ? c->err : g_create_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
}

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the KERNEL (per device), not to a context: several
// contexts share the generic kernel instances (and the fused spatial kernel whatever nx), each with its own
// shared-memory size, so the limit is only ever raised -- a context created later with a smaller grid must not
// lower it under the feet of an earlier one.
template <class F> cudaError_t smem_limit(F fn, size_t bytes)
{
    static std::mutex mu;
    static std::map<std::pair<int, const void *>, size_t> limit;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const void *key = reinterpret_cast<const void *>(fn);
    std::lock_guard<std::mutex> lock(mu);
    size_t &cur = limit[std::make_pair(dev, key)];
    if (bytes <= cur) return cudaSuccess;
    e = cudaFuncSetAttribute(key, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) cur = bytes;
    return e;
}

int cuda_fail(mphv_ctx *c, cudaError_t e, const char *what)
{
    set_err(c, "%s: %s", what, cudaGetErrorString(e));
    return MPHV_ERR_CUDA;
}

#define CUDA_TRY(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail((c), e_, #call); } while (0)

// Brackets one kernel launch with CUDA events when timing is on.
struct Timed {
    mphv_ctx *c; int slot; cudaEvent_t e0, e1; bool on;
    // alg_bytes: algorithmic (unfused) bytes of the launch; moved_bytes: what ONE pass must move (< 0: the same)
    Timed(mphv_ctx *c_, int slot_, double alg_bytes, double moved_bytes = -1.0) : c(c_), slot(slot_), e0(nullptr), e1(nullptr), on(false)
    {
        if (!c->timing) return;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { cudaGetLastError(); return; }
        on = true;
        c->slot_bytes[slot] = alg_bytes;
        c->slot_moved[slot] = moved_bytes < 0.0 ? alg_bytes : moved_bytes;
        cudaEventRecord(e0, c->stream);
    }
    ~Timed()
    {
        if (!on) return;
        cudaEventRecord(e1, c->stream);
        c->pending->push_back({ slot, e0, e1 });
    }
};

void drain_timing(mphv_ctx *c, bool keep)
{
    for (auto &p : *c->pending) {
        float ms = 0.f;
        if (keep && cudaEventElapsedTime(&ms, p.e0, p.e1) == cudaSuccess) {
            c->slot_ms[p.slot] += ms;
            c->slot_launches[p.slot]++;
        }
        cudaEventDestroy(p.e0); cudaEventDestroy(p.e1);
    }
    cudaGetLastError();
    c->pending->clear();
}

int after_launch(mphv_ctx *c, const char *what)
{
    c->launches++;
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(c, e, what); }
    return MPHV_OK;
}

// Makes the context's device current for the duration of one entry point and restores the caller's.
struct DevGuard {
    int prev; bool switched;
    explicit DevGuard(const mphv_ctx *c) : prev(-1), switched(false)
    {
        if (!c) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != c->dev) switched = cudaSetDevice(c->dev) == cudaSuccess;
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
};

bool is_finite(double x) { return x == x && !std::isinf(x); }

double host_vcentre(const mphv_ctx *c, int d, int j)
{
    return c->gd.vlo[d] + ((double)j + 0.5) * c->gd.dv[d];
}

// max over velocity cells of |s| for the spatial sweep d, s = (v dt)/dx evaluated as on the device
double max_courant_x(const mphv_ctx *c, int d, double dt)
{
    double m = 0.0;
    for (int j = 0; j < c->grid.nv[d]; ++j) {
        const double s = std::fabs((host_vcentre(c, d, j) * dt) / c->dx[d]);
        if (!(s == s)) return s;
        if (s > m) m = s;
    }
    return m;
}

double max_courant_v(const mphv_ctx *c, int d, double dt)
{
    return std::fabs((c->amax[d] * dt) / c->dv[d]);   // NaN propagates
}

// threads per CTA for kernels whose threads loop over the (vy, vx) plane of one spatial cell: the smallest
// multiple of 32 that covers the plane in the same number of rounds as 512 threads would (1600 -> 416, not 512)
int plane_block(long long plane)
{
    const long long rounds = (plane + 511) / 512;
    long long b = (plane + rounds - 1) / rounds;
    b = (b + 31) / 32 * 32;
    return (int)(b < 32 ? 32 : (b > 512 ? 512 : b));
}

unsigned grid_for(long long threads, int block) { return (unsigned)((threads + block - 1) / block); }

// ---- launchers ---------------------------------------------------------------------------

template <int KIND, int BC>
int launch_march(mphv_ctx *c, const MarchArgs &a)
{
    const int block = 256;
    Timed tm(c, KIND == KIND_SPACE ? SLOT_SX0 + a.dim : SLOT_VX + a.dim, 16.0 * (double)c->nf);
    if (a.inner % 2 == 0) {
        const long long threads = a.outer * (a.inner / 2);
        march2_kernel<2, 4, KIND, BC, false, 2><<<grid_for(threads, block), block, 0, c->stream>>>(a);
    } else {
        const long long threads = a.outer * a.inner;
        march2_kernel<1, 4, KIND, BC, false, 2><<<grid_for(threads, block), block, 0, c->stream>>>(a);
    }
    return after_launch(c, "march_kernel");
}

double *ws_moments(mphv_ctx *c) { return c->ws; }
double *ws_partials(mphv_ctx *c) { return c->ws + 10 * c->ns; }
double *ws_sum(mphv_ctx *c) { return c->ws + 10 * c->ns * (1 + (size_t)c->mom_tiles); }
double *ws_scalars(mphv_ctx *c) { return ws_sum(c) + SUM_BLOCKS; }

// V_vz with the moments of the new f accumulated in the same kernel (f read once less)
int launch_vz_moments(mphv_ctx *c, MarchArgs a, double *n, double *j, double *P)
{
    Timed tm(c, SLOT_VZMOM, 24.0 * (double)c->nf, 16.0 * (double)c->nf);
    a.mom = ws_partials(c);
    a.tiles = c->mom_tiles;
    a.per_tile = c->mom_per_tile;
    a.dV = c->dv[0] * c->dv[1] * c->dv[2];
    const unsigned grid = (unsigned)(c->ns * (size_t)c->mom_tiles);
    if (a.inner % 2 == 0) march2_kernel<2, 4, KIND_VEL, BC_WALL, true, 2><<<grid, c->mom_block, 0, c->stream>>>(a);
    else                  march2_kernel<1, 4, KIND_VEL, BC_WALL, true, 2><<<grid, c->mom_block, 0, c->stream>>>(a);
    int st = after_launch(c, "march_kernel(vz+moments)");
    if (st != MPHV_OK) return st;
    mom_finalize_kernel<<<grid_for((long long)c->ns * 10, 256), 256, 0, c->stream>>>(a.mom, c->mom_tiles, (long long)c->ns, a.dV, n, j, P);
    return after_launch(c, "mom_finalize_kernel");
}

int launch_vxy(mphv_ctx *c, double dt)
{
    PlaneArgs a;
    std::memset(&a, 0, sizeof a);
    a.f = c->f;
    a.planes = (long long)c->ns * c->grid.nv[2];
    a.nvx = c->grid.nv[0]; a.nvy = c->grid.nv[1]; a.nvz = c->grid.nv[2];
    a.hx = a.nvx / 2; a.hy = a.nvy / 2;
    a.inv_hx = 1.0f / (float)a.hx;
    a.dt = dt;
    a.E = c->E; a.B = c->B;
    a.g = c->gd;
    Timed tm(c, SLOT_VXY, 32.0 * (double)c->nf, 16.0 * (double)c->nf);
    const long long grid = a.planes < c->vxy_grid ? a.planes : c->vxy_grid;
    vxy_kernel<3><<<(unsigned)grid, c->vxy_T, c->vxy_smem, c->stream>>>(a);
    return after_launch(c, "vxy_kernel");
}

const int CUBE_NS = 4;                  // planes in flight per CTA (TMA ring depth), whole-V-stage kernel
const int PLANE_NS = 3;                 // same for the V_vx + V_vy variant (two CTAs per SM)

// The cube kernel is specialised for the velocity-plane shapes of the BASELINE.json configs
// (40x40, 32x32: compile-time row strides) and has a generic instance for everything else.
enum { CUBE_40 = 0, CUBE_32 = 1, CUBE_GEN = 2, CUBE_36 = 3, CUBE_16 = 4 };   // 36^3, 16^3: the paper's own velocity grids

template <bool MOM> void *cube_fn(int variant)
{
    switch (variant) {
    case CUBE_40: return (void *)vcube_kernel<CUBE_NS, true, MOM, 40, 40, 416, 1>;
    case CUBE_32: return (void *)vcube_kernel<CUBE_NS, true, MOM, 32, 32, 256, 2>;
    default:      return (void *)vcube_kernel<CUBE_NS, true, MOM, 0, 0, 512, 1>;
    }
}

// the same pipeline without the V_vz stage (V_vx + V_vy per plane)
void *plane_fn(int variant)
{
    switch (variant) {
    case CUBE_40: return (void *)vcube_kernel<PLANE_NS, false, false, 40, 40, 416, 2>;
    case CUBE_32: return (void *)vcube_kernel<PLANE_NS, false, false, 32, 32, 256, 3>;
    default:      return (void *)vcube_kernel<PLANE_NS, false, false, 0, 0, 512, 1>;
    }
}

// second-generation whole-V-stage kernel (mphv_vstage.cuh): same shape specialisations
template <bool MOM> void *vstage_fn(int variant)
{
    switch (variant) {
#ifndef MPHV_VS40_NS
#define MPHV_VS40_NS 3
#endif
    case CUBE_40: return (void *)vstage_kernel<MPHV_VS40_NS, MOM, 40, 40, 416, 1>;
#ifndef MPHV_VS32_NS
#define MPHV_VS32_NS 3          // measured on c2: ring depth 2 -> 3 and one 8-warp CTA per SM with up to 255 registers: 0.82 -> 0.67 ms
#define MPHV_VS32_MINB 1
#endif
    case CUBE_32: return (void *)vstage_kernel<MPHV_VS32_NS, MOM, 32, 32, 256, MPHV_VS32_MINB>;
    case CUBE_36: return (void *)vstage_kernel<3, MOM, 36, 36, 352, 1>;
#ifndef MPHV_VS16_MINB
#define MPHV_VS16_MINB 4         // measured at 256x128x16^3: 4 CTAs of 2 warps per SM with 255 registers beat 8 with 128 (0.75 vs 0.95 ms)
#endif
    case CUBE_16: return (void *)vstage_kernel<3, MOM, 16, 16, 64, MPHV_VS16_MINB>;
    default:      return (void *)vstage_kernel<3, MOM, 0, 0, 512, 1>;
    }
}
template <bool MOM> void *vstage_bs_fn(int variant)
{
    switch (variant) {
    case CUBE_40: return (void *)vstage_bs_kernel<MPHV_VS40_NS, MOM, 40, 40, 416, 1>;
    case CUBE_32: return (void *)vstage_bs_kernel<MPHV_VS32_NS, MOM, 32, 32, 256, MPHV_VS32_MINB>;
    case CUBE_36: return (void *)vstage_bs_kernel<3, MOM, 36, 36, 352, 1>;
    case CUBE_16: return (void *)vstage_bs_kernel<3, MOM, 16, 16, 64, MPHV_VS16_MINB>;
    default:      return (void *)vstage_bs_kernel<3, MOM, 0, 0, 512, 1>;
    }
}
// third-generation whole-V-stage kernel (mphv_vstage2.cuh): velocity planes of the BASELINE.json configs and of
// the paper's own grids. <ring depth, MOM, nvx, nvy, rows per patch, cells per run, threads, register-budget threads, CTAs per SM>
#ifndef MPHV_VS2_NS40
#define MPHV_VS2_NS40 3
#endif
template <bool MOM> void *vstage2_fn(int variant)
{
    switch (variant) {
    case CUBE_40: return (void *)vstage2_kernel<MPHV_VS2_NS40, MOM, 40, 40, 5, 10, 320, 384, 1>;
    case CUBE_32: return (void *)vstage2_kernel<3, MOM, 32, 32, 4, 8, 256, 256, 1>;
    case CUBE_36: return (void *)vstage2_kernel<3, MOM, 36, 36, 6, 12, 224, 256, 1>;
    case CUBE_16: return (void *)vstage2_kernel<3, MOM, 16, 16, 4, 8, 64, 64, 4>;
    default:      return nullptr;
    }
}
// fourth-generation whole-V-stage kernel (mphv_vstage3.cuh), warp-specialised:
// <ring depth, MOM, nvx, nvy, rows per patch, cells per run, B threads, launch threads, B registers, A registers>
#ifndef MPHV_VS3_NS40
#define MPHV_VS3_NS40 4
#endif
#ifndef MPHV_VS3_RB40
#define MPHV_VS3_RB40 144
#define MPHV_VS3_RA40 80
#endif
template <bool MOM> void *vstage3_fn(int variant)
{
    switch (variant) {
    case CUBE_40: return (void *)vstage3_kernel<MPHV_VS3_NS40, MOM, 40, 40, 5, 20, 320, 512, MPHV_VS3_RB40, MPHV_VS3_RA40>;
    // (32 x 32 planes: measured slower than vstage2_kernel, 0.72 vs 0.62 ms on c2 -- 8 B warps sit evenly on the schedulers there)
    default:      return nullptr;
    }
}
// the same roles with the three sweeps in face form (backsubstitution mode, mphv_vstage3_bs.cuh)
#ifndef MPHV_VS3BS_RB40
#define MPHV_VS3BS_RB40 144
#define MPHV_VS3BS_RA40 80
#endif
template <bool MOM> void *vstage3_bs_fn(int variant)
{
    switch (variant) {
    case CUBE_40: return (void *)vstage3_bs_kernel<MPHV_VS3_NS40, MOM, 40, 40, 5, 20, 320, 512, MPHV_VS3BS_RB40, MPHV_VS3BS_RA40>;
    default:      return nullptr;
    }
}
int vstage3_threads(int variant) { return variant == CUBE_40 ? 512 : 0; }
int vstage3_ns(int variant) { return variant == CUBE_40 ? MPHV_VS3_NS40 : 4; }
size_t vstage3_smem_bytes(int nvx, int nvy, int nvz, int ns)
{
    const size_t cells = (size_t)nvx * nvy, xcells = (size_t)nvx * (nvy + 4);
    return (ns * 2 * cells + 4 * 2 * xcells + nvz + 320) * sizeof(double) + (2 * ns + 8) * sizeof(uint64_t);
}

int vstage2_threads(int variant) { return variant == CUBE_40 ? 320 : variant == CUBE_32 ? 256 : variant == CUBE_36 ? 224 : variant == CUBE_16 ? 64 : 0; }
int vstage2_ns(int variant) { return variant == CUBE_40 ? MPHV_VS2_NS40 : 3; }
size_t vstage2_smem_bytes(int nvx, int nvy, int nvz, int ns)
{
    const size_t cells = (size_t)nvx * nvy, xcells = (size_t)nvx * (nvy + 4);
    return (ns * 2 * cells + VS_NXB * 2 * xcells + nvz + 320) * sizeof(double) + (ns + 2) * sizeof(uint64_t);
}

int vstage_ns(int variant) { return variant == CUBE_32 ? MPHV_VS32_NS : variant == CUBE_40 ? MPHV_VS40_NS : 3; }

size_t vstage_smem_bytes(int nvx, int nvy, int nvz, int ns, int T)
{
    const size_t cells = (size_t)nvx * nvy, xcells = (size_t)nvx * (nvy + 4);
    return (ns * 2 * cells + VS_NXB * 2 * xcells + nvz + 320 + 12 * (size_t)T) * sizeof(double) + (ns + 2) * sizeof(uint64_t);
}

size_t cube_smem_bytes(int nvx, int nvy, int nvz, int ns, bool reduce)
{
    const size_t cells = (size_t)nvx * nvy, xcells = (size_t)nvx * (nvy + 4);
    return (ns * cells + CUBE_NXB * xcells + CUBE_NT * 4 * (size_t)(nvx + nvy) + nvz + 6 * CUBE_FLD + (reduce ? 320 : 0)) * sizeof(double)
           + (ns + 2) * sizeof(uint64_t);
}

// V_vx, V_vy, V_vz (+ moments if n != NULL) in one pass over f; with_vz = false: V_vx, V_vy only
int launch_vcube(mphv_ctx *c, double dt, bool with_vz, double *n, double *j, double *P)
{
    CubeArgs a;
    std::memset(&a, 0, sizeof a);
    a.f = c->f;
    a.ns = (long long)c->ns;
    a.nvx = c->grid.nv[0]; a.nvy = c->grid.nv[1]; a.nvz = c->grid.nv[2];
    a.dt = dt;
    a.E = c->E; a.B = c->B;
    a.n = n; a.j = j; a.P = P;
    a.dV = c->dv[0] * c->dv[1] * c->dv[2];
    a.g = c->gd;
    Timed tm(c, !with_vz ? SLOT_VXY : n ? SLOT_VCUBE_MOM : SLOT_VCUBE, (!with_vz ? 32.0 : n ? 56.0 : 48.0) * (double)c->nf, 16.0 * (double)c->nf);
    void *fn = !with_vz ? plane_fn(c->cube_variant) : n ? cube_fn<true>(c->cube_variant) : cube_fn<false>(c->cube_variant);
    void *args[] = { &a };
    cudaError_t e = cudaLaunchKernel(fn, dim3((unsigned)(with_vz ? c->cube_grid : c->plane_grid)), dim3((unsigned)c->cube_T), args,
                                     with_vz ? c->cube_smem : c->plane_smem, c->stream);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(c, e, "vcube_kernel launch"); }
    return after_launch(c, "vcube_kernel");
}

// V_vx, V_vy, V_vz (+ moments if n != NULL) in one pass over f, two planes per pipeline iteration
int launch_vstage(mphv_ctx *c, double dt, double *n, double *j, double *P, bool backsub = false)
{
    const bool gen4 = c->vs_gen_max >= 4 && c->vs3_T > 0 && (!backsub || c->vs3_bs);
    const bool gen3 = c->vs_gen_max >= 3 && !backsub && !gen4 && c->vs2_T > 0;
    CubeArgs a;
    std::memset(&a, 0, sizeof a);
    a.f = c->f;
    a.ns = (long long)c->ns;
    a.nvx = c->grid.nv[0]; a.nvy = c->grid.nv[1]; a.nvz = c->grid.nv[2];
    a.dt = dt;
    a.E = c->E; a.B = c->B;
    a.n = n; a.j = j; a.P = P;
    a.dV = c->dv[0] * c->dv[1] * c->dv[2];
    a.sixth = 1.0 / 6.0;
    a.g = c->gd;
    Timed tm(c, n ? SLOT_VCUBE_MOM : SLOT_VCUBE, (n ? 56.0 : 48.0) * (double)c->nf, 16.0 * (double)c->nf);
    a.K = backsub ? c->bs_K : nullptr;
    void *fn = backsub && gen4 ? (n ? vstage3_bs_fn<true>(c->vs_variant) : vstage3_bs_fn<false>(c->vs_variant))
               : backsub ? (n ? vstage_bs_fn<true>(c->vs_variant) : vstage_bs_fn<false>(c->vs_variant))
               : gen4  ? (n ? vstage3_fn<true>(c->vs_variant) : vstage3_fn<false>(c->vs_variant))
               : gen3  ? (n ? vstage2_fn<true>(c->vs_variant) : vstage2_fn<false>(c->vs_variant))
                       : (n ? vstage_fn<true>(c->vs_variant) : vstage_fn<false>(c->vs_variant));
    void *args[] = { &a };
    cudaError_t e = gen4 ? cudaLaunchKernel(fn, dim3((unsigned)c->vs3_grid), dim3((unsigned)c->vs3_T), args, c->vs3_smem, c->stream)
                  : gen3 ? cudaLaunchKernel(fn, dim3((unsigned)c->vs2_grid), dim3((unsigned)c->vs2_T), args, c->vs2_smem, c->stream)
                         : cudaLaunchKernel(fn, dim3((unsigned)c->vs_grid), dim3((unsigned)c->vs_T), args, c->vs_smem, c->stream);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(c, e, "vstage_kernel launch"); }
    return after_launch(c, "vstage_kernel");
}

// S_x then S_y in one pass over f (mphv_sxy.cuh)
#ifndef MPHV_SXY_NR
#define MPHV_SXY_NR 6
#endif
const int SXY_NR = MPHV_SXY_NR;         // ring depth: SXY_NR - 1 rows in flight per CTA

enum { SXY_BCX_HALO = 2 };             // bcx argument of sxy_fn beyond MPHV_BC_PERIODIC / MPHV_BC_OUTFLOW
void *sxy_fn(int C, int bcx, int bcy)
{
#define SXY_ROW(CC, TM, MB, BX) \
    (bcy == MPHV_BC_PERIODIC ? (void *)sxy_kernel<CC, SXY_NR, BX, BC_PER, TM, MB> : (void *)sxy_kernel<CC, SXY_NR, BX, BC_OUT, TM, MB>)
#define SXY_PICK(CC, TM, MB) \
    (bcx == MPHV_BC_PERIODIC ? SXY_ROW(CC, TM, MB, BC_PER) : bcx == MPHV_BC_OUTFLOW ? SXY_ROW(CC, TM, MB, BC_OUT) : SXY_ROW(CC, TM, MB, BC_HALO))
    return C == 16 ? SXY_PICK(16, 512, 1) : SXY_PICK(8, 512, 1);
#undef SXY_PICK
#undef SXY_ROW
}

size_t sxy_smem_bytes(int C, int nx, int T, bool per_y)             // sized for the halo variant (nx + 4 cells per row)
{
    const size_t rowd = C == 16 ? sxy_row_doubles<16>(nx + 4) : sxy_row_doubles<8>(nx + 4);
    return (SXY_NR * rowd + (per_y ? 8 * (size_t)T : 0)) * sizeof(double);
}

int launch_sxy(mphv_ctx *c, double dt, bool halo = false, const double *lo = nullptr, const double *hi = nullptr)
{
    SxyArgs a;
    std::memset(&a, 0, sizeof a);
    a.f = c->f;
    a.nx = c->grid.nx[0]; a.ny = c->grid.nx[1];
    a.nvel = (long long)c->nvel;
    a.chunks = (int)(c->nvel / (size_t)c->sxy_C);
    a.dt = dt; a.dx = c->dx[0]; a.dy = c->dx[1];
    a.g = c->gd;
    Timed tm(c, SLOT_SXY, 32.0 * (double)c->nf, 16.0 * (double)c->nf);
    a.halo_lo = lo; a.halo_hi = hi;
    void *fn = sxy_fn(c->sxy_C, halo ? SXY_BCX_HALO : c->grid.bc[0], c->grid.bc[1]);
    void *args[] = { &a };
    const unsigned grid = (unsigned)((long long)c->grid.nx[2] * a.chunks);
    cudaError_t e = cudaLaunchKernel(fn, dim3(grid), dim3((unsigned)c->sxy_T), args, c->sxy_smem, c->stream);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(c, e, "sxy_kernel launch"); }
    return after_launch(c, "sxy_kernel");
}

MarchArgs march_args_space(const mphv_ctx *c, int d, double dt)
{
    MarchArgs a;
    std::memset(&a, 0, sizeof a);
    a.f = c->f;
    const long long nvel = (long long)c->nvel;
    const long long nx = c->grid.nx[0], ny = c->grid.nx[1], nz = c->grid.nx[2];
    if (d == 0)      { a.outer = nz * ny; a.inner = nvel; }
    else if (d == 1) { a.outer = nz;      a.inner = nx * nvel; }
    else             { a.outer = 1;       a.inner = ny * nx * nvel; }
    a.n = c->grid.nx[d];
    a.dim = d;
    a.dt = dt;
    a.dx = c->dx[d];
    a.g = c->gd;
    return a;
}

MarchArgs march_args_vel(const mphv_ctx *c, int d, double dt)
{
    MarchArgs a;
    std::memset(&a, 0, sizeof a);
    a.f = c->f;
    const long long nvx = c->grid.nv[0], nvy = c->grid.nv[1], nvz = c->grid.nv[2];
    if (d == 2) { a.outer = (long long)c->ns;       a.inner = nvy * nvx; }
    else        { a.outer = (long long)c->ns * nvz; a.inner = nvx; }
    a.n = c->grid.nv[d];
    a.dim = d;
    a.dt = dt;
    a.dx = c->dv[d];
    a.E = c->E; a.B = c->B;
    a.g = c->gd;
    return a;
}

int do_sweep_x(mphv_ctx *c, int d, double dt)
{
    MarchArgs a = march_args_space(c, d, dt);
    const double smax = max_courant_x(c, d, dt);
    if (c->grid.bc[d] == MPHV_BC_OUTFLOW) return launch_march<KIND_SPACE, BC_OUT>(c, a);
    if (smax < 1.0) return launch_march<KIND_SPACE, BC_PER>(c, a);
    // whole-cell shifts on a periodic axis: out of place through scratch, then copy back
    const long long threads = a.outer * a.inner;
    Timed tm(c, SLOT_SHIFT, 16.0 * (double)c->nf);
    shift_kernel<<<grid_for(threads, 256), 256, 0, c->stream>>>(a, c->f, c->scratch);
    int st = after_launch(c, "shift_kernel");
    if (st != MPHV_OK) return st;
    CUDA_TRY(c, cudaMemcpyAsync(c->f, c->scratch, c->nf * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    return MPHV_OK;
}

// ---- backsubstitution mode (mphv_backsub.cuh) ---------------------------------------------
// Coefficients and max |s_face| depend on (fields, dt): evaluated on the first use of a new dt
// (one kernel, 3 doubles to the host, one stream synchronisation), then cached.
int ensure_backsub(mphv_ctx *c, double dt)
{
    if (c->bs_valid && c->bs_dt == dt) return MPHV_OK;
    unsigned long long *smax = reinterpret_cast<unsigned long long *>(c->bs_K + 12 * c->ns);
    CUDA_TRY(c, cudaMemsetAsync(smax, 0, 3 * sizeof(unsigned long long), c->stream));
    int st;
    {
        Timed tm(c, SLOT_BSCOEF, 0.0);
        backsub_coeff_kernel<<<grid_for((long long)c->ns, 128), 128, 0, c->stream>>>(c->E, c->B, c->gd, dt, c->bs_K, smax);
        st = after_launch(c, "backsub_coeff_kernel");
    }
    if (st != MPHV_OK) return st;
    if (!c->deferred) {
        CUDA_TRY(c, cudaMemcpyAsync(c->bs_smax, smax, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    }
    c->bs_dt = dt; c->bs_valid = true;
    return MPHV_OK;
}

int do_sweep_v_backsub(mphv_ctx *c, int d)
{
    BacksubArgs a;
    a.f = c->f; a.K = c->bs_K; a.g = c->gd;
    const long long nvx = c->grid.nv[0], nvy = c->grid.nv[1], nvz = c->grid.nv[2];
    Timed tm(c, SLOT_VX + d, 16.0 * (double)c->nf);
    if (d == 0) {
        const long long rows = (long long)c->ns * nvz * nvy;
        const int block = 256;
        const int ch = (nvx % 4 == 0) ? 4 : (nvx % 2 == 0 ? 2 : 1);
        const int cpr = (int)(nvx / ch);
        if (cpr > block) { set_err(c, "nvx = %lld too large for the vx kernel (max %d)", nvx, block * 4); return MPHV_ERR_ARG; }
        const int rpc = block / cpr;
        const unsigned grid = (unsigned)((rows + rpc - 1) / rpc);
        if (ch == 4)      bs_vx_kernel<4><<<grid, block, 0, c->stream>>>(a, rows, rpc);
        else if (ch == 2) bs_vx_kernel<2><<<grid, block, 0, c->stream>>>(a, rows, rpc);
        else              bs_vx_kernel<1><<<grid, block, 0, c->stream>>>(a, rows, rpc);
        return after_launch(c, "bs_vx_kernel");
    }
    const long long outer = d == 2 ? (long long)c->ns : (long long)c->ns * nvz;
    const long long inner = d == 2 ? nvy * nvx : nvx;
    const int n = c->grid.nv[d];
    if (inner % 2 == 0) bs_march_kernel<2, 4><<<grid_for(outer * (inner / 2), 256), 256, 0, c->stream>>>(a, d, outer, n, inner);
    else                bs_march_kernel<1, 4><<<grid_for(outer * inner, 256), 256, 0, c->stream>>>(a, d, outer, n, inner);
    return after_launch(c, "bs_march_kernel");
}

int do_sweep_v(mphv_ctx *c, int d, double dt)
{
    if (c->vmode) return do_sweep_v_backsub(c, d);
    if (d == 0) {
        VxArgs a;
        std::memset(&a, 0, sizeof a);
        a.f = c->f;
        a.rows = (long long)c->ns * c->grid.nv[2] * c->grid.nv[1];
        a.nvx = c->grid.nv[0];
        a.dt = dt;
        a.E = c->E; a.B = c->B;
        a.g = c->gd;
        const int block = 256;
        const int ch = (a.nvx % 4 == 0) ? 4 : (a.nvx % 2 == 0 ? 2 : 1);
        const int cpr = a.nvx / ch;
        if (cpr > block) { set_err(c, "nvx = %d too large for the vx kernel (max %d)", a.nvx, block * 4); return MPHV_ERR_ARG; }
        a.rows_per_cta = block / cpr;
        const unsigned grid = (unsigned)((a.rows + a.rows_per_cta - 1) / a.rows_per_cta);
        Timed tm(c, SLOT_VX, 16.0 * (double)c->nf);
        if (ch == 4)      vx_kernel<4><<<grid, block, 0, c->stream>>>(a);
        else if (ch == 2) vx_kernel<2><<<grid, block, 0, c->stream>>>(a);
        else              vx_kernel<1><<<grid, block, 0, c->stream>>>(a);
        return after_launch(c, "vx_kernel");
    }
    MarchArgs a = march_args_vel(c, d, dt);
    return launch_march<KIND_VEL, BC_WALL>(c, a);
}

int do_moments(mphv_ctx *c, double *n, double *j, double *P);
int enqueue_range_flag(mphv_ctx *c, double dt);

// The whole V stage (active velocity sweeps in order vx, vy, vz) and, if n != NULL, the moments
// of the result. With fusion on: [vx+vy in one plane kernel], [vz + moments in one kernel].
int do_v_stage(mphv_ctx *c, double dt, double *n, double *j, double *P)
{
    int st;
    if (c->deferred && (st = enqueue_range_flag(c, dt)) != MPHV_OK) return st;
    const bool ax = c->grid.nv[0] > 1, ay = c->grid.nv[1] > 1, az = c->grid.nv[2] > 1;
    if (c->vmode && c->fusion >= 2 && c->vs_T > 0 && c->vs_bs) return launch_vstage(c, dt, n, j, P, true);
    if (c->vmode) {                                  // backsubstitution: three face-displaced sweeps, then the moments
        for (int d = 0; d < 3; ++d)
            if ((st = do_sweep_v_backsub(c, d)) != MPHV_OK) return st;
        return n ? do_moments(c, n, j, P) : MPHV_OK;
    }
    if (c->fusion >= 2 && c->vs_T > 0) return launch_vstage(c, dt, n, j, P);
    if (c->fusion >= 2 && c->cube_T > 0) return launch_vcube(c, dt, true, n, j, P);
    if (c->fusion && c->cube_T > 0 && c->plane_grid > 0) {
        if ((st = launch_vcube(c, dt, false, nullptr, nullptr, nullptr)) != MPHV_OK) return st;
    } else if (c->fusion && ax && ay && c->vxy_T > 0) {
        if ((st = launch_vxy(c, dt)) != MPHV_OK) return st;
    } else {
        if (ax && (st = do_sweep_v(c, 0, dt)) != MPHV_OK) return st;
        if (ay && (st = do_sweep_v(c, 1, dt)) != MPHV_OK) return st;
    }
    if (az && n && c->fusion) return launch_vz_moments(c, march_args_vel(c, 2, dt), n, j, P);
    if (az && (st = do_sweep_v(c, 2, dt)) != MPHV_OK) return st;
    if (n) return do_moments(c, n, j, P);
    return MPHV_OK;
}

int do_moments(mphv_ctx *c, double *n, double *j, double *P)
{
    MomArgs a;
    a.f = c->f; a.n = n; a.j = j; a.P = P;
    a.dV = c->dv[0] * c->dv[1] * c->dv[2];
    a.g = c->gd;
    const long long plane = (long long)c->grid.nv[0] * c->grid.nv[1];
    int block = 512;
    while (block > 32 && block / 2 >= plane) block /= 2;
    Timed tm(c, SLOT_MOM, 8.0 * (double)c->nf);
    moments_kernel<<<(unsigned)c->ns, block, 0, c->stream>>>(a);
    return after_launch(c, "moments_kernel");
}

int check_common(mphv_ctx *c, double dt, bool need_fields)
{
    if (!c) return MPHV_ERR_ARG;
    if (!is_finite(dt)) { set_err(c, "dt is not finite"); return MPHV_ERR_ARG; }
    if (!c->f) { set_err(c, "f not bound (mphv_bind_f)"); return MPHV_ERR_STATE; }
    if (need_fields && (!c->E || !c->B)) { set_err(c, "fields not set (mphv_set_fields)"); return MPHV_ERR_STATE; }
    return MPHV_OK;
}

int range_x(mphv_ctx *c, int d, double dt)
{
    const double smax = max_courant_x(c, d, dt);
    if (c->grid.bc[d] == MPHV_BC_OUTFLOW) {
        if (!(smax < 1.0)) { set_err(c, "spatial sweep %d: max |s| = %g >= 1 on an outflow axis", d, smax); return MPHV_ERR_RANGE; }
    } else if (!(smax < 1.0)) {
        if (!(smax == smax)) { set_err(c, "spatial sweep %d: Courant number is NaN", d); return MPHV_ERR_RANGE; }
        if (!c->scratch) { set_err(c, "spatial sweep %d: max |s| = %g >= 1 needs a scratch buffer", d, smax); return MPHV_ERR_RANGE; }
    }
    return MPHV_OK;
}

// deferred mode: one 1-thread kernel compares the device-resident bounds of all active velocity axes with 1
// and raises the sticky flag ws_scalars[4]
int enqueue_range_flag(mphv_ctx *c, double dt)
{
    int active = 0;
    for (int d = 0; d < 3; ++d) if (c->grid.nv[d] > 1) active |= 1 << d;
    const double *bound = c->vmode ? c->bs_K + 12 * c->ns : ws_scalars(c);
    range_flag_kernel<<<1, 32, 0, c->stream>>>(bound, dt, c->dv[0], c->dv[1], c->dv[2], active, c->vmode ? 0 : 1, ws_scalars(c) + 4);
    return after_launch(c, "range_flag_kernel");
}

int range_v(mphv_ctx *c, int d, double dt)
{
    if (c->deferred) {
        if (c->vmode) return ensure_backsub(c, dt);
        return MPHV_OK;                              // checked on the device (enqueue_range_flag)
    }
    if (c->vmode) {
        int st = ensure_backsub(c, dt);
        if (st != MPHV_OK) return st;
        if (!(c->bs_smax[d] < 1.0)) {
            set_err(c, "backsubstituted velocity sweep %d: max |s_face| = %g >= 1 (closed velocity box)", d, c->bs_smax[d]);
            return MPHV_ERR_RANGE;
        }
        return MPHV_OK;
    }
    // the fused kernels form s as fma(v, b, a) with dt / dv folded in: up to a few ulp away from (a dt) / dv
    const double smax = max_courant_v(c, d, dt) * (1.0 + 1.0e-15);
    if (!(smax < 1.0)) { set_err(c, "velocity sweep %d: max |s| = %g >= 1 (closed velocity box)", d, smax); return MPHV_ERR_RANGE; }
    return MPHV_OK;
}


// spatial sweeps along the axes below dmax, in order (dmax = 3: the whole X stage)
int x_stage(mphv_ctx *c, double dt, int dmax = 3)
{
    int st;
    int d0 = 0;
    if (dmax >= 2 && c->fusion >= 3 && c->sxy_T > 0 && max_courant_x(c, 0, dt) < 1.0 && max_courant_x(c, 1, dt) < 1.0) {
        if ((st = launch_sxy(c, dt)) != MPHV_OK) return st;        // S_x, S_y in one pass
        d0 = 2;
    }
    for (int d = d0; d < dmax; ++d)
        if (c->grid.nx[d] > 1 && (st = do_sweep_x(c, d, dt)) != MPHV_OK) return st;
    return MPHV_OK;
}


// ---- mphv_run_host as a slab pipeline ---------------------------------------------------------------
// f crosses PCIe both ways in one call; the step itself is ~40x shorter than either copy. The grid is cut
// into K slabs along its outermost active spatial axis (contiguous in memory); slab k is swept while slab
// k + 1 is still arriving and slab k - 1 is already leaving, so a call costs about max(H2D, D2H) instead of
// their sum. Every slab is a block of a spatial decomposition: sweeps along the lower axes and
// the V stage are local to it; the sweep along the slab axis takes its two ghost layers from the packed
// boundary layers of the neighbouring slabs (pack_halo_kernel, march2_kernel<BC_HALO>), packed AFTER the
// lower-axis sweeps of that slab and BEFORE its own slab-axis sweep overwrites them -- the order of the
// multi-GPU path (halo.py). Result: that of mphv_step on the whole grid up to fp64 rounding.

void destroy_pipe(mphv_ctx *c)
{
    HostPipe *hp = c->pipe;
    if (!hp) return;
    for (mphv_ctx *s : hp->sub) if (s) mphv_destroy(s);
    for (cudaEvent_t e : hp->ev_in) if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : hp->ev_out) if (e) cudaEventDestroy(e);
    if (hp->h2d) cudaStreamDestroy(hp->h2d);
    if (hp->d2h) cudaStreamDestroy(hp->d2h);
    if (hp->halo) cudaFree(hp->halo);
    if (hp->fld) cudaFree(hp->fld);
    if (hp->mom) cudaFree(hp->mom);
    cudaGetLastError();
    delete hp;
    c->pipe = nullptr;
}

// builds the slab contexts once; false = this grid is not pipelined (the caller takes the plain path)
bool ensure_pipe(mphv_ctx *c)
{
    if (c->pipe) return true;
    if (c->pipe_failed) return false;
    int axis = -1;
    for (int d = 2; d >= 0; --d) if (c->grid.nx[d] > 1) { axis = d; break; }
    if (axis < 0) return false;
    const int n = c->grid.nx[axis];
    int K = n / 4 < 16 ? n / 4 : 16;
    if (K < 3 || c->nf * sizeof(double) < (size_t)16 << 20) return false;      // small problems: not worth it
    HostPipe *hp = new (std::nothrow) HostPipe();
    if (!hp) return false;
    c->pipe = hp;
    hp->axis = axis; hp->K = K;
    hp->halo = hp->fld = hp->mom = nullptr; hp->h2d = hp->d2h = nullptr;
    hp->layer = c->nf / (size_t)n;
    hp->row0.resize(K + 1);
    for (int k = 0; k <= K; ++k) hp->row0[k] = (int)((long long)n * k / K);
    hp->sub.assign(K, nullptr); hp->ev_in.assign(K, nullptr); hp->ev_out.assign(K, nullptr);
    bool ok = cudaStreamCreateWithFlags(&hp->h2d, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&hp->d2h, cudaStreamNonBlocking) == cudaSuccess;
    size_t nsk_max = 0;
    for (int k = 0; k < K && ok; ++k) {
        mphv_grid g = c->grid;
        mphv_box b = c->box;
        const int nk = hp->row0[k + 1] - hp->row0[k];
        g.nx[axis] = nk;
        b.xlo[axis] = c->box.xlo[axis] + c->dx[axis] * hp->row0[k];
        b.xhi[axis] = c->box.xlo[axis] + c->dx[axis] * hp->row0[k + 1];
        mphv_ctx *s = mphv_create(&g, &b, c->qm);
        ok = s != nullptr;
        if (!ok) break;
        s->dx[axis] = c->dx[axis];                       // bitwise the parent's cell width (Courant numbers)
        hp->sub[k] = s;
        if (s->ns > nsk_max) nsk_max = s->ns;
        ok = cudaEventCreateWithFlags(&hp->ev_in[k], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&hp->ev_out[k], cudaEventDisableTiming) == cudaSuccess;
    }
    if (ok) {
        hp->halo_stride = 2 * hp->layer;
        ok = cudaMalloc(&hp->halo, (size_t)K * 2 * hp->halo_stride * sizeof(double)) == cudaSuccess &&
             cudaMalloc(&hp->fld, 6 * c->ns * sizeof(double)) == cudaSuccess &&
             cudaMalloc(&hp->mom, 10 * nsk_max * sizeof(double)) == cudaSuccess;
    }
    if (!ok) { cudaGetLastError(); destroy_pipe(c); c->pipe_failed = true; return false; }
    return true;
}

// One full split step of the bound f, slab by slab. f_in: host source of f (NULL: f is already on the device);
// f_out: host destination (NULL: f stays); mn/mj/mP: full-grid moment arrays on the device or NULL.
int pipe_step(mphv_ctx *c, double dt, const double *f_in, double *f_out, double *mn, double *mj, double *mP)
{
    HostPipe *hp = c->pipe;
    const int K = hp->K, axis = hp->axis;
    const bool periodic = c->grid.bc[axis] == MPHV_BC_PERIODIC;
    int st;
    // per-slab views of f and of the fields ([3][ns_k] blocks cut out of the parent's [3][ns])
    size_t off_cells = 0;
    for (int k = 0; k < K; ++k) {
        mphv_ctx *s = hp->sub[k];
        s->stream = c->stream; s->fusion = c->fusion; s->vs_gen_max = c->vs_gen_max; s->timing = 0; s->vmode = 0;
        s->f = c->f + (size_t)hp->row0[k] * hp->layer; s->scratch = nullptr;
        double *Ek = hp->fld + 6 * off_cells, *Bk = Ek + 3 * s->ns;
        CUDA_TRY(c, cudaMemcpy2DAsync(Ek, s->ns * sizeof(double), c->E + off_cells, c->ns * sizeof(double), s->ns * sizeof(double), 3, cudaMemcpyDeviceToDevice, c->stream));
        CUDA_TRY(c, cudaMemcpy2DAsync(Bk, s->ns * sizeof(double), c->B + off_cells, c->ns * sizeof(double), s->ns * sizeof(double), 3, cudaMemcpyDeviceToDevice, c->stream));
        s->E = Ek; s->B = Bk; s->deferred = false;
        for (int d = 0; d < 3; ++d) s->amax[d] = c->amax[d];          // the parent's bound covers every slab
        off_cells += s->ns;
    }
    if (f_in) {
        cudaEvent_t ready = hp->ev_out[0];               // f must be free (earlier work on the compute stream done)
        CUDA_TRY(c, cudaEventRecord(ready, c->stream));
        CUDA_TRY(c, cudaStreamWaitEvent(hp->h2d, ready, 0));
        for (int k = 0; k < K; ++k) {
            const size_t o = (size_t)hp->row0[k] * hp->layer, cnt = hp->sub[k]->nf;
            CUDA_TRY(c, cudaMemcpyAsync(c->f + o, f_in + o, cnt * sizeof(double), cudaMemcpyHostToDevice, hp->h2d));
            CUDA_TRY(c, cudaEventRecord(hp->ev_in[k], hp->h2d));
        }
    }
    auto lo_buf = [&](int k) { return hp->halo + (size_t)(2 * k) * hp->halo_stride; };       // packed LOW layers of slab k
    auto hi_buf = [&](int k) { return hp->halo + (size_t)(2 * k + 1) * hp->halo_stride; };   // packed HIGH layers of slab k
    // lower-axis sweeps of slab k, then its two boundary layers packed for the neighbours
    auto stage_local = [&](int k) -> int {
        mphv_ctx *s = hp->sub[k];
        if (f_in) CUDA_TRY(c, cudaStreamWaitEvent(c->stream, hp->ev_in[k], 0));
        int e = x_stage(s, dt, axis);
        if (e != MPHV_OK) return e;
        if ((e = mphv_pack_halo(s, axis, 0, lo_buf(k))) != MPHV_OK) return e;
        return mphv_pack_halo(s, axis, 1, hi_buf(k));
    };
    // slab-axis sweep with the neighbours' layers, V stage, moments, and the way out
    auto stage_rest = [&](int k) -> int {
        mphv_ctx *s = hp->sub[k];
        const double *lo = k > 0 ? hi_buf(k - 1) : (periodic ? hi_buf(K - 1) : nullptr);
        const double *hi = k + 1 < K ? lo_buf(k + 1) : (periodic ? lo_buf(0) : nullptr);
        MarchArgs a = march_args_space(s, axis, dt);
        a.halo_lo = lo; a.halo_hi = hi;
        int e = launch_march<KIND_SPACE, BC_HALO>(s, a);
        if (e != MPHV_OK) return e;
        if (mn) {
            double *tn = hp->mom, *tj = tn + s->ns, *tP = tn + 4 * s->ns;
            if ((e = do_v_stage(s, dt, tn, tj, tP)) != MPHV_OK) return e;
            const size_t o = (size_t)hp->row0[k] * (c->ns / (size_t)c->grid.nx[axis]);
            const size_t w = s->ns * sizeof(double), dp = c->ns * sizeof(double);
            CUDA_TRY(c, cudaMemcpyAsync(mn + o, tn, w, cudaMemcpyDeviceToDevice, c->stream));
            CUDA_TRY(c, cudaMemcpy2DAsync(mj + o, dp, tj, w, w, 3, cudaMemcpyDeviceToDevice, c->stream));
            CUDA_TRY(c, cudaMemcpy2DAsync(mP + o, dp, tP, w, w, 6, cudaMemcpyDeviceToDevice, c->stream));
        } else if ((e = do_v_stage(s, dt, nullptr, nullptr, nullptr)) != MPHV_OK) return e;
        if (f_out) {
            const size_t o = (size_t)hp->row0[k] * hp->layer;
            CUDA_TRY(c, cudaEventRecord(hp->ev_out[k], c->stream));
            CUDA_TRY(c, cudaStreamWaitEvent(hp->d2h, hp->ev_out[k], 0));
            CUDA_TRY(c, cudaMemcpyAsync(f_out + o, c->f + o, s->nf * sizeof(double), cudaMemcpyDeviceToHost, hp->d2h));
        }
        return MPHV_OK;
    };
    // order: local(0), local(1), rest(0) [outflow] ..., a periodic axis keeps slab 0 for last (it needs slab K-1)
    if ((st = stage_local(0)) != MPHV_OK) return st;
    for (int k = 1; k < K; ++k) {
        if ((st = stage_local(k)) != MPHV_OK) return st;
        if (k - 1 > 0 || !periodic) { if ((st = stage_rest(k - 1)) != MPHV_OK) return st; }
    }
    if (periodic) {
        // slab K-1 needs lo_buf(0) (packed), slab 0 needs hi_buf(K-1) (packed): both are there now
        if ((st = stage_rest(K - 1)) != MPHV_OK) return st;
        if ((st = stage_rest(0)) != MPHV_OK) return st;
    } else if ((st = stage_rest(K - 1)) != MPHV_OK) return st;
    for (int k = 0; k < K; ++k) c->launches += hp->sub[k]->launches, hp->sub[k]->launches = 0;
    if (f_out) {                                         // the compute stream's owner waits for the copies out
        cudaEvent_t done = hp->ev_in[0];
        CUDA_TRY(c, cudaEventRecord(done, hp->d2h));
        CUDA_TRY(c, cudaStreamWaitEvent(c->stream, done, 0));
    }
    return MPHV_OK;
}

bool pipe_eligible(mphv_ctx *c, double dt)
{
    if (c->vmode || c->deferred) return false;
    int axis = -1;
    for (int d = 2; d >= 0; --d) if (c->grid.nx[d] > 1) { axis = d; break; }
    if (axis < 0 || !(max_courant_x(c, axis, dt) < 1.0)) return false;      // halo sweeps need |s| < 1
    // the slabs have no scratch buffer (s->scratch = nullptr): a whole-cell shift (|s| >= 1 on a lower, periodic
    // axis, which the parent accepts when it has one) must take the plain path
    for (int d = 0; d < axis; ++d)
        if (c->grid.nx[d] > 1 && !(max_courant_x(c, d, dt) < 1.0)) return false;
    return ensure_pipe(c);
}

}  // namespace

extern "C" {

// for the other translation unit of the library (mphv_coupled.cu): text of mphv_last_error(NULL)
void mphv_internal_set_create_error(const char *text) { set_err(nullptr, "%s", text ? text : ""); }

// for mphv_plasma_destroy: a species whose fields still are the plasma's centred-field buffers (bound by
// mphv_set_fields_deferred inside mphv_plasma_step) loses them before that buffer is freed, so that its next
// sweep fails with MPHV_ERR_STATE instead of reading freed memory. Fields the caller bound since are left alone.
void mphv_internal_unbind_fields(mphv_ctx *c, const double *E, const double *B)
{
    if (!c || c->E != E || c->B != B) return;
    c->E = c->B = nullptr;
    c->deferred = false;
    c->bs_valid = false;
    for (int d = 0; d < 3; ++d) c->amax[d] = 0.0;
}

mphv_ctx *mphv_create(const mphv_grid *grid, const mphv_box *box, double q_over_m)
{
    if (!grid || !box) { set_err(nullptr, "grid or box is NULL"); return nullptr; }
    if (!is_finite(q_over_m)) { set_err(nullptr, "q_over_m is not finite"); return nullptr; }
    for (int d = 0; d < 3; ++d) {
        if (grid->nx[d] < 1 || grid->nv[d] < 1) { set_err(nullptr, "extent < 1 in dimension %d", d); return nullptr; }
        if ((grid->nx[d] > 1 && grid->nx[d] < 4) || (grid->nv[d] > 1 && grid->nv[d] < 4)) {
            set_err(nullptr, "active extent < 4 in dimension %d", d); return nullptr;
        }
        if (grid->bc[d] != MPHV_BC_PERIODIC && grid->bc[d] != MPHV_BC_OUTFLOW) { set_err(nullptr, "bad bc[%d]", d); return nullptr; }
        if (grid->nx[d] > 1 && !(box->xhi[d] > box->xlo[d] && is_finite(box->xhi[d]) && is_finite(box->xlo[d]))) {
            set_err(nullptr, "xhi <= xlo in dimension %d", d); return nullptr;
        }
        if (grid->nv[d] > 1 && !(box->vhi[d] > box->vlo[d] && is_finite(box->vhi[d]) && is_finite(box->vlo[d]))) {
            set_err(nullptr, "vhi <= vlo in dimension %d", d); return nullptr;
        }
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { set_err(nullptr, "no CUDA device: %s (there is no CPU fallback)", cudaGetErrorString(e)); cudaGetLastError(); return nullptr; }
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) { set_err(nullptr, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e)); cudaGetLastError(); return nullptr; }
    if (major != 10) { set_err(nullptr, "%s: device compute capability %d.x, need 10.x (sm_100a)", mphv_strerror(MPHV_ERR_ARCH), major); return nullptr; }

    mphv_ctx *c = new (std::nothrow) mphv_ctx;
    if (!c) { set_err(nullptr, "out of host memory"); return nullptr; }
    std::memset(c, 0, sizeof *c);
    c->pending = new (std::nothrow) std::vector<mphv_ctx::Pending>();
    if (!c->pending) { set_err(nullptr, "out of host memory"); delete c; return nullptr; }
    c->dev = dev;
    c->grid = *grid; c->box = *box; c->qm = q_over_m;
    c->ns = (size_t)grid->nx[0] * grid->nx[1] * grid->nx[2];
    c->nvel = (size_t)grid->nv[0] * grid->nv[1] * grid->nv[2];
    c->nf = c->ns * c->nvel;
    c->fusion = 3;
    c->vs_gen_max = 4;
    for (int d = 0; d < 3; ++d) {
        c->dx[d] = grid->nx[d] > 1 ? (box->xhi[d] - box->xlo[d]) / (double)grid->nx[d] : 1.0;
        c->dv[d] = grid->nv[d] > 1 ? (box->vhi[d] - box->vlo[d]) / (double)grid->nv[d] : 1.0;
        c->gd.nx[d] = grid->nx[d]; c->gd.nv[d] = grid->nv[d];
        c->gd.dv[d] = c->dv[d];
        c->gd.vlo[d] = grid->nv[d] > 1 ? box->vlo[d] : -0.5;
        c->amax[d] = NAN;
    }
    c->gd.qm = q_over_m;
    c->gd.ns = (long long)c->ns;
    c->gd.nvel = (long long)c->nvel;
    {   // CTA tiling of the fused V_vz + moments kernel: tiles of <= 256 (vector) pencils per spatial cell
        const long long plane = (long long)grid->nv[0] * grid->nv[1];
        const long long innerV = plane % 2 == 0 ? plane / 2 : plane;
        c->mom_tiles = (int)((innerV + 255) / 256);
        c->mom_per_tile = (int)((innerV + c->mom_tiles - 1) / c->mom_tiles);
        c->mom_block = ((c->mom_per_tile + 31) / 32) * 32;
    }
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    c->vxy_T = 0;
    if (grid->nv[0] >= 4 && grid->nv[1] >= 4 && grid->nv[0] % 2 == 0 && grid->nv[1] % 2 == 0) {
        const int nvx = grid->nv[0], nvy = grid->nv[1];
        int T = ((nvx / 2) * (nvy / 2) + 31) / 32 * 32;
        const int T2 = (nvx + nvy + 31) / 32 * 32;
        if (T < T2) T = T2;
        if (T > 448) T = 448;
        const size_t smem = ((size_t)(3 + 1) * nvx * nvy + 6 * (size_t)(nvx + nvy) + 3) * sizeof(double);
        int max_optin = 0;
        cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (nvx + nvy <= T && smem <= (size_t)max_optin &&
            smem_limit(vxy_kernel<3>, smem) == cudaSuccess) {
            int per_sm = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, vxy_kernel<3>, T, smem) == cudaSuccess && per_sm > 0) {
                c->vxy_T = T; c->vxy_smem = smem; c->vxy_grid = per_sm * c->sm_count;
            }
        }
        cudaGetLastError();
    }
    c->cube_T = 0;
    if (grid->nv[0] % 4 == 0 && grid->nv[1] % 4 == 0 && grid->nv[2] >= 4) {
        const int nvx = grid->nv[0], nvy = grid->nv[1], nvz = grid->nv[2];
        const int items = nvy * (nvx / 4);
        const int T = (items + 31) / 32 * 32;
        const int variant = (nvx == 40 && nvy == 40) ? CUBE_40 : (nvx == 32 && nvy == 32) ? CUBE_32 : CUBE_GEN;
        const size_t smem = cube_smem_bytes(nvx, nvy, nvz, CUBE_NS, true);
        const size_t psmem = cube_smem_bytes(nvx, nvy, nvz, PLANE_NS, false);
        int max_optin = 0;
        cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (T <= 512 && nvx + nvy <= T && smem <= (size_t)max_optin &&
            smem_limit(cube_fn<true>(variant), smem) == cudaSuccess &&
            smem_limit(cube_fn<false>(variant), smem) == cudaSuccess) {
            int per_sm = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cube_fn<true>(variant), T, smem) == cudaSuccess && per_sm > 0) {
                long long g = (long long)per_sm * c->sm_count;
                const long long gmin = ((long long)c->ns + CUBE_FLD - 1) / CUBE_FLD;   // <= CUBE_FLD cells per CTA
                if (g < gmin) g = ((gmin + c->sm_count - 1) / c->sm_count) * c->sm_count;
                if (g > (long long)c->ns) g = (long long)c->ns;
                c->cube_T = T; c->cube_smem = smem; c->cube_grid = (int)g; c->cube_variant = variant;
                c->plane_grid = 0;
                if (smem_limit(plane_fn(variant), psmem) == cudaSuccess &&
                    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, plane_fn(variant), T, psmem) == cudaSuccess && per_sm > 0) {
                    long long pg = (long long)per_sm * c->sm_count;
                    if (pg < gmin) pg = ((gmin + c->sm_count - 1) / c->sm_count) * c->sm_count;
                    if (pg > (long long)c->ns) pg = (long long)c->ns;
                    c->plane_grid = (int)pg; c->plane_smem = psmem;
                }
            }
        }
        cudaGetLastError();
    }
    c->vs_T = 0;
    if (grid->nv[0] % 4 == 0 && grid->nv[1] % 4 == 0 && grid->nv[2] >= 4 && grid->nv[2] % 2 == 0) {
        const int nvx = grid->nv[0], nvy = grid->nv[1], nvz = grid->nv[2];
        const int T = (nvy * (nvx / 4) + 31) / 32 * 32;
        const int variant = (nvx == 40 && nvy == 40) ? CUBE_40 : (nvx == 32 && nvy == 32) ? CUBE_32
                          : (nvx == 36 && nvy == 36) ? CUBE_36 : (nvx == 16 && nvy == 16) ? CUBE_16 : CUBE_GEN;
        const size_t smem = vstage_smem_bytes(nvx, nvy, nvz, vstage_ns(variant), T);
        int max_optin = 0, per_sm = 0;
        cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (T <= 512 && smem <= (size_t)max_optin &&
            smem_limit(vstage_fn<true>(variant), smem) == cudaSuccess &&
            smem_limit(vstage_fn<false>(variant), smem) == cudaSuccess &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, vstage_fn<true>(variant), T, smem) == cudaSuccess && per_sm > 0) {
            long long g = (long long)per_sm * c->sm_count;
            if (g > (long long)c->ns) g = (long long)c->ns;
            c->vs_T = T; c->vs_smem = smem; c->vs_grid = (int)g; c->vs_variant = variant;
            c->vs_bs = smem_limit(vstage_bs_fn<true>(variant), smem) == cudaSuccess &&
                       smem_limit(vstage_bs_fn<false>(variant), smem) == cudaSuccess;
        }
        cudaGetLastError();
        c->vs3_T = 0;
        if (c->vs_T > 0 && vstage3_fn<true>(variant)) {
            const size_t smem3 = vstage3_smem_bytes(nvx, nvy, nvz, vstage3_ns(variant));
            const int T3 = vstage3_threads(variant);
            int per3 = 0;
            if (smem3 <= (size_t)max_optin &&
                smem_limit(vstage3_fn<true>(variant), smem3) == cudaSuccess &&
                smem_limit(vstage3_fn<false>(variant), smem3) == cudaSuccess &&
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per3, vstage3_fn<true>(variant), T3, smem3) == cudaSuccess && per3 > 0) {
                long long g3 = (long long)c->sm_count;
                if (g3 > (long long)c->ns) g3 = (long long)c->ns;
                c->vs3_T = T3; c->vs3_smem = smem3; c->vs3_grid = (int)g3;
                c->vs3_bs = vstage3_bs_fn<true>(variant) &&
                            smem_limit(vstage3_bs_fn<true>(variant), smem3) == cudaSuccess &&
                            smem_limit(vstage3_bs_fn<false>(variant), smem3) == cudaSuccess;
            }
            cudaGetLastError();
        }
        c->vs2_T = 0;
        if (c->vs_T > 0 && vstage2_fn<true>(variant)) {
            const size_t smem2 = vstage2_smem_bytes(nvx, nvy, nvz, vstage2_ns(variant));
            const int T2 = vstage2_threads(variant);
            int per2 = 0;
            if (smem2 <= (size_t)max_optin &&
                smem_limit(vstage2_fn<true>(variant), smem2) == cudaSuccess &&
                smem_limit(vstage2_fn<false>(variant), smem2) == cudaSuccess &&
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per2, vstage2_fn<true>(variant), T2, smem2) == cudaSuccess && per2 > 0) {
                long long g2 = (long long)per2 * c->sm_count;
                if (g2 > (long long)c->ns) g2 = (long long)c->ns;
                c->vs2_T = T2; c->vs2_smem = smem2; c->vs2_grid = (int)g2;
            }
            cudaGetLastError();
        }
    }
    c->sxy_T = 0;
    if (grid->nx[0] >= 8 && grid->nx[0] % 4 == 0 && grid->nx[1] >= 4) {
        const int nx = grid->nx[0];
        int C = 0;
#ifndef MPHV_SXY_PREFER_C8
        if (c->nvel % 16 == 0 && (nx / 4) * 16 <= 512) C = 16;
        else
#endif
        if (c->nvel % 8 == 0 && (nx / 4) * 8 <= 512) C = 8;
        if (C) {
            const int T = (nx / 4) * C;
            size_t smem = 0;
            int max_optin = 0;
            cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
            bool ok = true;
            for (int by = 0; by < 2 && ok; ++by) {
                const size_t sm = sxy_smem_bytes(C, nx, T, by == MPHV_BC_PERIODIC);
                if (by == grid->bc[1]) smem = sm;
                for (int bx = 0; bx < 3 && ok; ++bx)
                    ok = sm <= (size_t)max_optin &&
                         smem_limit(sxy_fn(C, bx, by), sm) == cudaSuccess;
            }
            if (ok) { c->sxy_T = T; c->sxy_C = C; c->sxy_smem = smem; }
        }
        cudaGetLastError();
    }
    e = cudaMalloc(&c->ws, (10 * c->ns * (1 + (size_t)c->mom_tiles) + SUM_BLOCKS + 8) * sizeof(double));
    if (e != cudaSuccess) { set_err(nullptr, "cudaMalloc workspace: %s", cudaGetErrorString(e)); cudaGetLastError(); delete c->pending; delete c; return nullptr; }
    return c;
}

int mphv_destroy(mphv_ctx *c)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (c->ws) cudaFree(c->ws);
    if (c->fld) cudaFree(c->fld);
    if (c->bs_K) cudaFree(c->bs_K);
    destroy_pipe(c);
    if (c->pending) { drain_timing(c, false); delete c->pending; }
    delete c;
    return MPHV_OK;
}

int mphv_set_stream(mphv_ctx *c, void *s)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    c->stream = (cudaStream_t)s;
    return MPHV_OK;
}

size_t mphv_f_count(const mphv_ctx *c) { return c ? c->nf : 0; }
size_t mphv_space_count(const mphv_ctx *c) { return c ? c->ns : 0; }

int mphv_bind_f(mphv_ctx *c, double *f, double *scratch)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!f) { set_err(c, "f_dev is NULL"); return MPHV_ERR_ARG; }
    if (((uintptr_t)f & 15) || ((uintptr_t)scratch & 15)) { set_err(c, "f/scratch must be 16-byte aligned"); return MPHV_ERR_ARG; }
    if (scratch == f) { set_err(c, "scratch must not alias f"); return MPHV_ERR_ARG; }
    c->f = f; c->scratch = scratch;
    return MPHV_OK;
}

int mphv_set_fields_deferred(mphv_ctx *c, const double *E, const double *B)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!E || !B) { set_err(c, "E_dev or B_dev is NULL"); return MPHV_ERR_ARG; }
    int st;
    {
        Timed tm(c, SLOT_AMAX, 0.0);
        amax_kernel<<<1, 1024, 0, c->stream>>>(E, B, c->gd, ws_scalars(c));
        st = after_launch(c, "amax_kernel");
    }
    if (st != MPHV_OK) return st;
    if (!c->deferred) CUDA_TRY(c, cudaMemsetAsync(ws_scalars(c) + 4, 0, sizeof(double), c->stream));
    c->E = E; c->B = B;
    c->bs_valid = false;
    c->deferred = true;
    for (int d = 0; d < 3; ++d) c->amax[d] = NAN;
    return MPHV_OK;
}

int mphv_deferred_status(mphv_ctx *c)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!c->deferred) return MPHV_OK;
    double flag = 0.0;
    CUDA_TRY(c, cudaMemcpyAsync(&flag, ws_scalars(c) + 4, sizeof flag, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    if (flag != 0.0) {
        CUDA_TRY(c, cudaMemsetAsync(ws_scalars(c) + 4, 0, sizeof(double), c->stream));
        set_err(c, "a velocity sweep enqueued since the last query had |s| >= 1 (deferred RANGE check): f is lost");
        return MPHV_ERR_RANGE;
    }
    return MPHV_OK;
}

int mphv_set_fields(mphv_ctx *c, const double *E, const double *B)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!E || !B) { set_err(c, "E_dev or B_dev is NULL"); return MPHV_ERR_ARG; }
    double *out = ws_scalars(c);
    int st;
    {
        Timed tm(c, SLOT_AMAX, 0.0);
        amax_kernel<<<1, 1024, 0, c->stream>>>(E, B, c->gd, out);
        st = after_launch(c, "amax_kernel");
    }
    if (st != MPHV_OK) return st;
    c->deferred = false;
    double h[3];
    CUDA_TRY(c, cudaMemcpyAsync(h, out, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->E = E; c->B = B;
    c->bs_valid = false;
    for (int d = 0; d < 3; ++d) c->amax[d] = h[d];
    return MPHV_OK;
}

int mphv_sweep_x(mphv_ctx *c, int dim, double dt)
{
    DevGuard dg(c);
    int st = check_common(c, dt, false);
    if (st != MPHV_OK) return st;
    if (dim < 0 || dim > 2 || c->grid.nx[dim] < 2) { set_err(c, "spatial dim %d out of range or inactive", dim); return MPHV_ERR_ARG; }
    st = range_x(c, dim, dt);
    if (st != MPHV_OK) return st;
    return do_sweep_x(c, dim, dt);
}

int mphv_sweep_v(mphv_ctx *c, int dim, double dt)
{
    DevGuard dg(c);
    int st = check_common(c, dt, true);
    if (st != MPHV_OK) return st;
    if (dim < 0 || dim > 2 || c->grid.nv[dim] < 2) { set_err(c, "velocity dim %d out of range or inactive", dim); return MPHV_ERR_ARG; }
    st = range_v(c, dim, dt);
    if (st != MPHV_OK) return st;
    if (c->deferred && (st = enqueue_range_flag(c, dt)) != MPHV_OK) return st;
    return do_sweep_v(c, dim, dt);
}

static int step_checks(mphv_ctx *c, double dt)
{
    int st = check_common(c, dt, true);
    if (st != MPHV_OK) return st;
    for (int d = 0; d < 3; ++d)
        if (c->grid.nx[d] > 1 && (st = range_x(c, d, dt)) != MPHV_OK) return st;
    for (int d = 0; d < 3; ++d)
        if (c->grid.nv[d] > 1 && (st = range_v(c, d, dt)) != MPHV_OK) return st;
    return MPHV_OK;
}

static int step_impl(mphv_ctx *c, double dt, double *n, double *j, double *P)
{
    int st = step_checks(c, dt);
    if (st != MPHV_OK) return st;
    if ((st = x_stage(c, dt)) != MPHV_OK) return st;
    return do_v_stage(c, dt, n, j, P);
}

int mphv_step(mphv_ctx *c, double dt)
{
    DevGuard dg(c);
    return step_impl(c, dt, nullptr, nullptr, nullptr);
}

int mphv_moments(mphv_ctx *c, double *n, double *j, double *P)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!n || !j || !P) { set_err(c, "n_dev, j_dev or P_dev is NULL"); return MPHV_ERR_ARG; }
    if (!c->f) { set_err(c, "f not bound (mphv_bind_f)"); return MPHV_ERR_STATE; }
    return do_moments(c, n, j, P);
}

int mphv_stage_x(mphv_ctx *c, double dt)
{
    DevGuard dg(c);
    int st = check_common(c, dt, false);
    if (st != MPHV_OK) return st;
    for (int d = 0; d < 3; ++d)
        if (c->grid.nx[d] > 1 && (st = range_x(c, d, dt)) != MPHV_OK) return st;
    return x_stage(c, dt);
}

int mphv_stage_v(mphv_ctx *c, double dt, double *n, double *j, double *P)
{
    DevGuard dg(c);
    int st = check_common(c, dt, true);
    if (st != MPHV_OK) return st;
    if (n && (!j || !P)) { set_err(c, "n_dev given but j_dev or P_dev is NULL"); return MPHV_ERR_ARG; }
    for (int d = 0; d < 3; ++d)
        if (c->grid.nv[d] > 1 && (st = range_v(c, d, dt)) != MPHV_OK) return st;
    return do_v_stage(c, dt, n, j, P);
}

size_t mphv_halo_count(const mphv_ctx *c, int dim)
{
    if (!c || dim < 0 || dim > 2 || c->grid.nx[dim] < 2) return 0;
    return 2 * (c->nf / (size_t)c->grid.nx[dim]);
}

int mphv_pack_halo(mphv_ctx *c, int dim, int side, double *buf)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (dim < 0 || dim > 2 || c->grid.nx[dim] < 2) { set_err(c, "spatial dim %d out of range or inactive", dim); return MPHV_ERR_ARG; }
    if (side != 0 && side != 1) { set_err(c, "side must be 0 (low end) or 1 (high end)"); return MPHV_ERR_ARG; }
    if (!buf || ((uintptr_t)buf & 15)) { set_err(c, "buf_dev is NULL or not 16-byte aligned"); return MPHV_ERR_ARG; }
    if (!c->f) { set_err(c, "f not bound (mphv_bind_f)"); return MPHV_ERR_STATE; }
    const MarchArgs a = march_args_space(c, dim, 0.0);
    const int row0 = side ? a.n - 2 : 0;
    Timed tm(c, SLOT_PACK, 2.0 * 8.0 * (double)mphv_halo_count(c, dim));
    if (a.inner % 2 == 0)
        pack_halo_kernel<2><<<grid_for(a.outer * 2 * (a.inner / 2), 256), 256, 0, c->stream>>>(c->f, buf, a.outer, a.n, a.inner, row0);
    else
        pack_halo_kernel<1><<<grid_for(a.outer * 2 * a.inner, 256), 256, 0, c->stream>>>(c->f, buf, a.outer, a.n, a.inner, row0);
    return after_launch(c, "pack_halo_kernel");
}

int mphv_sweep_x_halo(mphv_ctx *c, int dim, double dt, const double *lo, const double *hi)
{
    DevGuard dg(c);
    int st = check_common(c, dt, false);
    if (st != MPHV_OK) return st;
    if (dim < 0 || dim > 2 || c->grid.nx[dim] < 2) { set_err(c, "spatial dim %d out of range or inactive", dim); return MPHV_ERR_ARG; }
    if (((uintptr_t)lo & 15) || ((uintptr_t)hi & 15)) { set_err(c, "halo buffers must be 16-byte aligned"); return MPHV_ERR_ARG; }
    if (c->grid.bc[dim] == MPHV_BC_PERIODIC && (!lo || !hi)) {
        set_err(c, "spatial sweep %d: a periodic axis needs both halo buffers", dim); return MPHV_ERR_ARG;
    }
    const double smax = max_courant_x(c, dim, dt);
    if (!(smax < 1.0)) { set_err(c, "spatial sweep %d with halos: max |s| = %g >= 1 reaches past the two boundary cells", dim, smax); return MPHV_ERR_RANGE; }
    MarchArgs a = march_args_space(c, dim, dt);
    a.halo_lo = lo; a.halo_hi = hi;
    return launch_march<KIND_SPACE, BC_HALO>(c, a);
}

int mphv_maxwellian(mphv_ctx *c, size_t count, const double *n, const double *j, const double *P, double *f_out)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!n || !j || !P || !f_out) { set_err(c, "n_dev, j_dev, P_dev or f_out_dev is NULL"); return MPHV_ERR_ARG; }
    if (count == 0) return MPHV_OK;
    if (count > 0x7fffffffu) { set_err(c, "count too large"); return MPHV_ERR_ARG; }
    MaxwArgs a;
    a.n = n; a.j = j; a.P = P; a.count = (long long)count; a.f_out = f_out; a.g = c->gd;
    Timed tm(c, SLOT_MAXW, 8.0 * (double)count * (double)c->nvel);
    maxwellian_kernel<<<(unsigned)count, 256, 0, c->stream>>>(a);
    return after_launch(c, "maxwellian_kernel");
}

int mphv_exchange_maxwellian(mphv_ctx *c, int dim, int side, const double *n_fl, const double *j_fl, const double *P_fl)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (dim < 0 || dim > 2 || c->grid.nx[dim] < 4) { set_err(c, "spatial dim %d out of range or inactive", dim); return MPHV_ERR_ARG; }
    if (side != 0 && side != 1) { set_err(c, "side must be 0 (low end) or 1 (high end)"); return MPHV_ERR_ARG; }
    if (!n_fl || !j_fl || !P_fl) { set_err(c, "n_fl_dev, j_fl_dev or P_fl_dev is NULL"); return MPHV_ERR_ARG; }
    if (!c->f) { set_err(c, "f not bound (mphv_bind_f)"); return MPHV_ERR_STATE; }
    const long long sstride[3] = { 1, c->grid.nx[0], (long long)c->grid.nx[0] * c->grid.nx[1] };
    const int da = dim == 0 ? 1 : 0, db = dim == 2 ? 1 : 2;
    ExchArgs a;
    a.f = c->f; a.n_fl = n_fl; a.j_fl = j_fl; a.P_fl = P_fl;
    a.plane = (long long)(c->ns / (size_t)c->grid.nx[dim]);
    a.sa = sstride[da]; a.sb = sstride[db]; a.sd = sstride[dim];
    a.na = c->grid.nx[da]; a.n = c->grid.nx[dim]; a.side = side; a.g = c->gd;
    const int block = plane_block((long long)c->grid.nv[0] * c->grid.nv[1]);
    Timed tm(c, SLOT_EXCH, 2.0 * (double)a.plane * 16.0 * (double)c->nvel);
    exchange_kernel<<<(unsigned)(2 * a.plane), block, 0, c->stream>>>(a);
    return after_launch(c, "exchange_kernel");
}

int mphv_match_moments(mphv_ctx *c, const double *n_t, const double *j_t, const double *P_t)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!n_t || !j_t || !P_t) { set_err(c, "n_t_dev, j_t_dev or P_t_dev is NULL"); return MPHV_ERR_ARG; }
    if (!c->f) { set_err(c, "f not bound (mphv_bind_f)"); return MPHV_ERR_STATE; }
    MatchArgs a;
    a.f = c->f; a.n_t = n_t; a.j_t = j_t; a.P_t = P_t; a.g = c->gd;
    const int block = plane_block((long long)c->grid.nv[0] * c->grid.nv[1]);
    Timed tm(c, SLOT_MATCH, 24.0 * (double)c->nf);
    match_kernel<<<(unsigned)c->ns, block, 0, c->stream>>>(a);
    return after_launch(c, "match_kernel");
}

int mphv_stage_x_halo(mphv_ctx *c, double dt, const double *lo, const double *hi)
{
    DevGuard dg(c);
    int st = check_common(c, dt, false);
    if (st != MPHV_OK) return st;
    if (c->grid.nx[0] < 2) { set_err(c, "spatial dim 0 is inactive"); return MPHV_ERR_ARG; }
    if (((uintptr_t)lo & 15) || ((uintptr_t)hi & 15)) { set_err(c, "halo buffers must be 16-byte aligned"); return MPHV_ERR_ARG; }
    if (c->grid.bc[0] == MPHV_BC_PERIODIC && (!lo || !hi)) {
        set_err(c, "stage_x_halo: a periodic x axis needs both halo buffers"); return MPHV_ERR_ARG;
    }
    if (!(max_courant_x(c, 0, dt) < 1.0)) {
        set_err(c, "spatial sweep 0 with halos: max |s| = %g >= 1 reaches past the two boundary cells", max_courant_x(c, 0, dt));
        return MPHV_ERR_RANGE;
    }
    for (int d = 1; d < 3; ++d)
        if (c->grid.nx[d] > 1 && (st = range_x(c, d, dt)) != MPHV_OK) return st;
    int d0 = 1;
    if (c->fusion >= 3 && c->sxy_T > 0 && c->grid.nx[1] > 1 && max_courant_x(c, 1, dt) < 1.0) {
        if ((st = launch_sxy(c, dt, true, lo, hi)) != MPHV_OK) return st;          // S_x (ghosts from the slabs), S_y
        d0 = 2;
    } else {
        MarchArgs a = march_args_space(c, 0, dt);
        a.halo_lo = lo; a.halo_hi = hi;
        if ((st = launch_march<KIND_SPACE, BC_HALO>(c, a)) != MPHV_OK) return st;
    }
    for (int d = d0; d < 3; ++d)
        if (c->grid.nx[d] > 1 && (st = do_sweep_x(c, d, dt)) != MPHV_OK) return st;
    return MPHV_OK;
}

int mphv_step_moments(mphv_ctx *c, double dt, double *n, double *j, double *P)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!n || !j || !P) { set_err(c, "n_dev, j_dev or P_dev is NULL"); return MPHV_ERR_ARG; }
    return step_impl(c, dt, n, j, P);
}

int mphv_run_host(mphv_ctx *c, double *f_host, int nsteps, double dt, double *n_host, double *j_host, double *P_host)
{
    DevGuard dg(c);
    int st = step_checks(c, dt);
    if (st != MPHV_OK) return st;
    if (!f_host || nsteps < 0) { set_err(c, "f_host is NULL or nsteps < 0"); return MPHV_ERR_ARG; }
    double *mn = ws_moments(c), *mj = mn + c->ns, *mP = mn + 4 * c->ns;
    if (nsteps > 0 && pipe_eligible(c, dt)) {
        // slab pipeline: the first step overlaps the copy in, the last one the copy out (see HostPipe)
        for (int s = 0; s < nsteps; ++s) {
            const bool first = s == 0, last = s + 1 == nsteps;
            if (first || last) st = pipe_step(c, dt, first ? f_host : nullptr, last ? f_host : nullptr,
                                              last ? mn : nullptr, last ? mj : nullptr, last ? mP : nullptr);
            else st = mphv_step(c, dt);
            if (st != MPHV_OK) return st;
        }
    } else {
        CUDA_TRY(c, cudaMemcpyAsync(c->f, f_host, c->nf * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        for (int s = 0; s + 1 < nsteps; ++s)
            if ((st = mphv_step(c, dt)) != MPHV_OK) return st;
        if (nsteps > 0) st = step_impl(c, dt, mn, mj, mP);       // last step with the moments fused in
        else st = do_moments(c, mn, mj, mP);
        if (st != MPHV_OK) return st;
        CUDA_TRY(c, cudaMemcpyAsync(f_host, c->f, c->nf * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    }
    if (n_host) CUDA_TRY(c, cudaMemcpyAsync(n_host, mn, c->ns * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    if (j_host) CUDA_TRY(c, cudaMemcpyAsync(j_host, mj, 3 * c->ns * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    if (P_host) CUDA_TRY(c, cudaMemcpyAsync(P_host, mP, 6 * c->ns * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    if (c->deferred) return mphv_deferred_status(c);      // synchronises; a context left in deferred mode reports its RANGE flag here
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MPHV_OK;
}

int mphv_step_fields_host(mphv_ctx *c, const double *E_host, const double *B_host, double dt,
                          double *n_host, double *j_host, double *P_host)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!E_host || !B_host || !n_host || !j_host || !P_host) { set_err(c, "a host pointer is NULL"); return MPHV_ERR_ARG; }
    if (!c->f) { set_err(c, "f not bound (mphv_bind_f)"); return MPHV_ERR_STATE; }
    if (!c->fld) {
        cudaError_t e = cudaMalloc(&c->fld, 6 * c->ns * sizeof(double));
        if (e != cudaSuccess) { c->fld = nullptr; return cuda_fail(c, e, "cudaMalloc field staging"); }
    }
    CUDA_TRY(c, cudaMemcpyAsync(c->fld, E_host, 3 * c->ns * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->fld + 3 * c->ns, B_host, 3 * c->ns * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    // the Courant bound of the new fields stays on the device: the call's one synchronisation is the one at its end
    int st = mphv_set_fields_deferred(c, c->fld, c->fld + 3 * c->ns);
    if (st != MPHV_OK) return st;
    double *mn = ws_moments(c), *mj = mn + c->ns, *mP = mn + 4 * c->ns;
    if ((st = step_impl(c, dt, mn, mj, mP)) != MPHV_OK) return st;
    CUDA_TRY(c, cudaMemcpyAsync(n_host, mn, c->ns * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(j_host, mj, 3 * c->ns * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(P_host, mP, 6 * c->ns * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    return mphv_deferred_status(c);                  // synchronises; MPHV_ERR_RANGE if a velocity sweep had |s| >= 1
}

int mphv_sum_f(mphv_ctx *c, double *sum_dev)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (!sum_dev) { set_err(c, "sum_dev is NULL"); return MPHV_ERR_ARG; }
    if (!c->f) { set_err(c, "f not bound (mphv_bind_f)"); return MPHV_ERR_STATE; }
    double *partial = ws_sum(c);
    Timed tm(c, SLOT_SUM, 8.0 * (double)c->nf);
    sum_kernel<<<SUM_BLOCKS, 256, 0, c->stream>>>(c->f, (long long)c->nf, partial);
    int st = after_launch(c, "sum_kernel");
    if (st != MPHV_OK) return st;
    sum_kernel<<<1, 256, 0, c->stream>>>(partial, SUM_BLOCKS, sum_dev);
    return after_launch(c, "sum_kernel(final)");
}

int mphv_set_timing(mphv_ctx *c, int enabled)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    drain_timing(c, false);
    for (int i = 0; i < 24; ++i) { c->slot_ms[i] = 0.0; c->slot_launches[i] = 0; c->slot_bytes[i] = 0.0; c->slot_moved[i] = 0.0; }
    c->timing = enabled ? 1 : 0;
    return MPHV_OK;
}

int mphv_timing_slots(void) { return SLOT_COUNT; }

int mphv_get_timing(mphv_ctx *c, int slot, char *name, size_t name_cap, double *total_ms,
                    uint64_t *launches, double *alg_bytes_per_launch)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (slot < 0 || slot >= SLOT_COUNT) { set_err(c, "timing slot %d out of range", slot); return MPHV_ERR_ARG; }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    drain_timing(c, true);
    if (name && name_cap) { std::strncpy(name, SLOT_NAMES[slot], name_cap - 1); name[name_cap - 1] = 0; }
    if (total_ms) *total_ms = c->slot_ms[slot];
    if (launches) *launches = c->slot_launches[slot];
    if (alg_bytes_per_launch) *alg_bytes_per_launch = c->slot_bytes[slot];
    return MPHV_OK;
}

int mphv_get_timing_moved(mphv_ctx *c, int slot, double *moved_bytes_per_launch)
{
    if (!c) return MPHV_ERR_ARG;
    if (slot < 0 || slot >= SLOT_COUNT || !moved_bytes_per_launch) { set_err(c, "timing slot %d out of range or NULL output", slot); return MPHV_ERR_ARG; }
    *moved_bytes_per_launch = c->slot_moved[slot];
    return MPHV_OK;
}

uint64_t mphv_launch_count(const mphv_ctx *c) { return c ? c->launches : 0; }

int mphv_set_vmode(mphv_ctx *c, int mode)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    if (mode != MPHV_V_PLAIN && mode != MPHV_V_BACKSUB) { set_err(c, "vmode must be MPHV_V_PLAIN or MPHV_V_BACKSUB"); return MPHV_ERR_ARG; }
    if (mode == MPHV_V_BACKSUB) {
        if (c->grid.nv[0] < 2 || c->grid.nv[1] < 2 || c->grid.nv[2] < 2) {
            set_err(c, "backsubstitution needs all three velocity dimensions active"); return MPHV_ERR_ARG;
        }
        if (!c->bs_K) {
            cudaError_t e = cudaMalloc(&c->bs_K, (12 * c->ns + 4) * sizeof(double));
            if (e != cudaSuccess) { c->bs_K = nullptr; return cuda_fail(c, e, "cudaMalloc backsubstitution coefficients"); }
        }
    }
    c->vmode = mode;
    c->bs_valid = false;
    return MPHV_OK;
}

int mphv_set_fusion(mphv_ctx *c, int enabled)
{
    DevGuard dg(c);
    if (!c) return MPHV_ERR_ARG;
    c->fusion = enabled < 0 ? 0 : (enabled > 3 ? 3 : enabled);
    return MPHV_OK;
}

int mphv_set_vstage_generation(mphv_ctx *c, int generation)
{
    if (!c) return MPHV_ERR_ARG;
    if (generation < 2 || generation > 4) { set_err(c, "whole-V-stage kernel generation must be 2, 3 or 4"); return MPHV_ERR_ARG; }
    c->vs_gen_max = generation;
    return MPHV_OK;
}

const char *mphv_strerror(int code)
{
    switch (code) {
    case MPHV_OK: return "MPHV_OK";
    case MPHV_ERR_ARG: return "MPHV_ERR_ARG: bad argument";
    case MPHV_ERR_STATE: return "MPHV_ERR_STATE: f or fields not bound";
    case MPHV_ERR_RANGE: return "MPHV_ERR_RANGE: Courant number out of range for this axis";
    case MPHV_ERR_CUDA: return "MPHV_ERR_CUDA: CUDA runtime error";
    case MPHV_ERR_ARCH: return "MPHV_ERR_ARCH: device is not sm_100";
    default: return "unknown mphv status";
    }
}

const char *mphv_last_error(const mphv_ctx *c) { return c ? c->err : g_create_err; }

}  // extern "C"
