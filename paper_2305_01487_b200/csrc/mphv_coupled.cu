// mphv_coupled.cu -- C-ABI of the field solver (mphv_maxwell_*) and of the coupled multi-species step
// (mphv_plasma_*), include/mphv.h "closing the loop". The species are driven through the public C ABI only
// (mphv_set_stream, mphv_set_fields_deferred, mphv_step_moments, mphv_moments); the field arithmetic runs in the
// kernels of mphv_fields.cuh. No CPU fallback.
#include "../../include/mphv.h"
#include "mphv_fields.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

using namespace mphv;

struct mphv_maxwell {
    mphv_field_grid grid;
    FieldDev gd;
    int dev;
    cudaStream_t stream;
    double *E, *B;
    char err[512];
};

struct mphv_plasma {
    mphv_maxwell *m;
    int ns_species;
    mphv_ctx *sp[FLD_MAX_SPECIES];
    double q[FLD_MAX_SPECIES];
    size_t ns;
    int dev;
    int concurrent;
    bool have_moments;
    cudaStream_t sstream[FLD_MAX_SPECIES];      // one stream per species (concurrent mode)
    cudaEvent_t ev_mom[FLD_MAX_SPECIES], ev_fields;
    double *buf;                                // [nspecies][10 ns] moments | [3 ns] J | [3 ns] Ec | [3 ns] Bc
    char err[512];
};

// defined in mphv.cu (same library): the text buffer mphv_last_error(NULL) returns
extern "C" void mphv_internal_set_create_error(const char *text);
extern "C" void mphv_internal_unbind_fields(mphv_ctx *c, const double *E, const double *B);

namespace {

const long long FUSED_MAX_CELLS = 65536;

void fail_create(const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    mphv_internal_set_create_error(buf);
}

template <class T> int fail(T *o, int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(o->err, sizeof o->err, fmt, ap);
    va_end(ap);
    return code;
}

template <class T> int cuda_fail(T *o, cudaError_t e, const char *what)
{
    return fail(o, MPHV_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

#define FLD_TRY(o, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cudaGetLastError(); return cuda_fail((o), e_, #call); } } while (0)

struct DevGuard2 {
    int prev; bool switched;
    explicit DevGuard2(int dev) : prev(-1), switched(false)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DevGuard2() { if (switched) cudaSetDevice(prev); }
};

int launched(mphv_maxwell *m, const char *what)
{
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(m, e, what); }
    return MPHV_OK;
}

unsigned blocks(long long n) { return (unsigned)((n + 255) / 256); }

MaxwellArgs base_args(const mphv_maxwell *m)
{
    MaxwellArgs a;
    std::memset(&a, 0, sizeof a);
    a.g = m->gd; a.E = m->E; a.B = m->B;
    return a;
}

int need_fields(mphv_maxwell *m)
{
    if (!m) return MPHV_ERR_ARG;
    if (!m->E || !m->B) return fail(m, MPHV_ERR_STATE, "fields not bound (mphv_maxwell_bind)");
    return MPHV_OK;
}

// [J = sum q_s j_s ->] reps x Maxwell(dt; J) [-> centred fields]: one launch on small grids
int maxwell_run(mphv_maxwell *m, const MaxwellArgs &a0)
{
    MaxwellArgs a = a0;
    if (a.g.ns <= FUSED_MAX_CELLS) {
        maxwell_fused_kernel<<<1, 1024, 0, m->stream>>>(a);
        return launched(m, "maxwell_fused_kernel");
    }
    int st;
    if (a.Jout) {
        current_kernel<<<blocks(3 * a.g.ns), 256, 0, m->stream>>>(a);
        if ((st = launched(m, "current_kernel")) != MPHV_OK) return st;
        a.J = a.Jout;
    }
    for (int r = 0; r < a.reps; ++r) {
        faraday_kernel<<<blocks(a.g.ns), 256, 0, m->stream>>>(a, 0.5 * a.dt);
        if ((st = launched(m, "faraday_kernel")) != MPHV_OK) return st;
        ampere_kernel<<<blocks(a.g.ns), 256, 0, m->stream>>>(a, a.dt);
        if ((st = launched(m, "ampere_kernel")) != MPHV_OK) return st;
        faraday_kernel<<<blocks(a.g.ns), 256, 0, m->stream>>>(a, 0.5 * a.dt);
        if ((st = launched(m, "faraday_kernel")) != MPHV_OK) return st;
    }
    if (a.Ec) {
        centre_kernel<<<blocks(a.g.ns), 256, 0, m->stream>>>(a);
        if ((st = launched(m, "centre_kernel")) != MPHV_OK) return st;
    }
    return MPHV_OK;
}

bool is_fin(double x) { return x == x && !std::isinf(x); }

double *mom_n(mphv_plasma *p, int s) { return p->buf + (size_t)s * 10 * p->ns; }
double *buf_J(mphv_plasma *p) { return p->buf + (size_t)p->ns_species * 10 * p->ns; }
double *buf_Ec(mphv_plasma *p) { return buf_J(p) + 3 * p->ns; }
double *buf_Bc(mphv_plasma *p) { return buf_J(p) + 6 * p->ns; }

}  // namespace

extern "C" {

mphv_maxwell *mphv_maxwell_create(const mphv_field_grid *g)
{
    if (!g) { fail_create("field grid is NULL"); return nullptr; }
    for (int d = 0; d < 3; ++d) {
        if (g->nx[d] < 1) { fail_create("extent < 1 in dimension %d", d); return nullptr; }
        if (g->bc[d] != MPHV_BC_PERIODIC && g->bc[d] != MPHV_BC_OUTFLOW) { fail_create("bad bc[%d]", d); return nullptr; }
        if (g->nx[d] > 1 && !(g->dx[d] > 0.0 && is_fin(g->dx[d]))) { fail_create("dx[%d] must be positive", d); return nullptr; }
    }
    if (!is_fin(g->c2) || !is_fin(g->inv_eps0) || g->c2 < 0.0) { fail_create("c2 / inv_eps0 not finite"); return nullptr; }
    int dev = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) { fail_create("no CUDA device: %s (there is no CPU fallback)", cudaGetErrorString(e)); cudaGetLastError(); return nullptr; }
    if (major != 10) { fail_create("device compute capability %d.x, need 10.x (sm_100a)", major); return nullptr; }
    mphv_maxwell *m = new (std::nothrow) mphv_maxwell;
    if (!m) { fail_create("out of host memory"); return nullptr; }
    std::memset(m, 0, sizeof *m);
    m->grid = *g;
    m->dev = dev;
    m->gd.ns = 1;
    for (int d = 0; d < 3; ++d) {
        m->gd.nx[d] = g->nx[d]; m->gd.bc[d] = g->bc[d];
        m->gd.inv_dx[d] = g->nx[d] > 1 ? 1.0 / g->dx[d] : 0.0;
        m->gd.ns *= g->nx[d];
    }
    m->gd.c2 = g->c2; m->gd.inv_eps0 = g->inv_eps0;
    return m;
}

int mphv_maxwell_destroy(mphv_maxwell *m)
{
    if (!m) return MPHV_ERR_ARG;
    delete m;
    return MPHV_OK;
}

int mphv_maxwell_set_stream(mphv_maxwell *m, void *s)
{
    if (!m) return MPHV_ERR_ARG;
    m->stream = (cudaStream_t)s;
    return MPHV_OK;
}

int mphv_maxwell_bind(mphv_maxwell *m, double *E, double *B)
{
    if (!m) return MPHV_ERR_ARG;
    if (!E || !B) return fail(m, MPHV_ERR_ARG, "E_dev or B_dev is NULL");
    m->E = E; m->B = B;
    return MPHV_OK;
}

int mphv_maxwell_faraday(mphv_maxwell *m, double dt)
{
    int st = need_fields(m);
    if (st != MPHV_OK) return st;
    if (!is_fin(dt)) return fail(m, MPHV_ERR_ARG, "dt is not finite");
    DevGuard2 dg(m->dev);
    faraday_kernel<<<blocks(m->gd.ns), 256, 0, m->stream>>>(base_args(m), dt);
    return launched(m, "faraday_kernel");
}

int mphv_maxwell_ampere(mphv_maxwell *m, const double *J, double dt)
{
    int st = need_fields(m);
    if (st != MPHV_OK) return st;
    if (!is_fin(dt)) return fail(m, MPHV_ERR_ARG, "dt is not finite");
    DevGuard2 dg(m->dev);
    MaxwellArgs a = base_args(m);
    a.J = J;
    ampere_kernel<<<blocks(m->gd.ns), 256, 0, m->stream>>>(a, dt);
    return launched(m, "ampere_kernel");
}

int mphv_maxwell_step(mphv_maxwell *m, const double *J, double dt)
{
    int st = need_fields(m);
    if (st != MPHV_OK) return st;
    if (!is_fin(dt)) return fail(m, MPHV_ERR_ARG, "dt is not finite");
    DevGuard2 dg(m->dev);
    MaxwellArgs a = base_args(m);
    a.J = J; a.dt = dt; a.reps = 1;
    return maxwell_run(m, a);
}

int mphv_maxwell_centre(mphv_maxwell *m, double *Ec, double *Bc)
{
    int st = need_fields(m);
    if (st != MPHV_OK) return st;
    if (!Ec || !Bc) return fail(m, MPHV_ERR_ARG, "Ec_dev or Bc_dev is NULL");
    DevGuard2 dg(m->dev);
    MaxwellArgs a = base_args(m);
    a.Ec = Ec; a.Bc = Bc;
    centre_kernel<<<blocks(m->gd.ns), 256, 0, m->stream>>>(a);
    return launched(m, "centre_kernel");
}

int mphv_maxwell_current(mphv_maxwell *m, int nspecies, const double *q, const double *const *j, double *J)
{
    if (!m) return MPHV_ERR_ARG;
    if (nspecies < 1 || nspecies > FLD_MAX_SPECIES) return fail(m, MPHV_ERR_ARG, "nspecies must be 1..%d", (int)FLD_MAX_SPECIES);
    if (!q || !j || !J) return fail(m, MPHV_ERR_ARG, "q_host, j_dev_ptrs or J_dev is NULL");
    DevGuard2 dg(m->dev);
    MaxwellArgs a = base_args(m);
    a.nspecies = nspecies; a.Jout = J;
    for (int s = 0; s < nspecies; ++s) {
        if (!j[s]) return fail(m, MPHV_ERR_ARG, "j_dev_ptrs[%d] is NULL", s);
        a.q[s] = q[s]; a.j[s] = j[s];
    }
    current_kernel<<<blocks(3 * m->gd.ns), 256, 0, m->stream>>>(a);
    return launched(m, "current_kernel");
}

const char *mphv_maxwell_last_error(const mphv_maxwell *m) { return m ? m->err : mphv_last_error(nullptr); }

// --------------------------------------------------------------------------------------------- plasma

mphv_plasma *mphv_plasma_create(mphv_maxwell *m, int nspecies, mphv_ctx *const *species, const double *q)
{
    if (!m || !species || !q) { fail_create("maxwell, species or q_host is NULL"); return nullptr; }
    if (nspecies < 1 || nspecies > FLD_MAX_SPECIES) { fail_create("nspecies must be 1..%d", (int)FLD_MAX_SPECIES); return nullptr; }
    for (int s = 0; s < nspecies; ++s) {
        if (!species[s]) { fail_create("species[%d] is NULL", s); return nullptr; }
        if (mphv_space_count(species[s]) != (size_t)m->gd.ns) {
            fail_create("species %d has %zu spatial cells, the field solver %lld", s, mphv_space_count(species[s]), m->gd.ns);
            return nullptr;
        }
        if (!is_fin(q[s])) { fail_create("q_host[%d] is not finite", s); return nullptr; }
    }
    mphv_plasma *p = new (std::nothrow) mphv_plasma;
    if (!p) { fail_create("out of host memory"); return nullptr; }
    std::memset(p, 0, sizeof *p);
    p->m = m; p->ns_species = nspecies; p->ns = (size_t)m->gd.ns; p->dev = m->dev; p->concurrent = 0;
    DevGuard2 dg(p->dev);
    for (int s = 0; s < nspecies; ++s) { p->sp[s] = species[s]; p->q[s] = q[s]; }
    cudaError_t e = cudaMalloc(&p->buf, ((size_t)nspecies * 10 + 9) * p->ns * sizeof(double));
    for (int s = 0; s < nspecies && e == cudaSuccess; ++s) {
        e = cudaStreamCreateWithFlags(&p->sstream[s], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_mom[s], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_fields, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        fail_create("mphv_plasma_create: %s", cudaGetErrorString(e));
        cudaGetLastError();
        mphv_plasma_destroy(p);
        return nullptr;
    }
    return p;
}

int mphv_plasma_destroy(mphv_plasma *p)
{
    if (!p) return MPHV_ERR_ARG;
    DevGuard2 dg(p->dev);
    cudaDeviceSynchronize();
    for (int s = 0; s < p->ns_species; ++s) {
        if (p->sp[s]) mphv_set_stream(p->sp[s], p->m->stream);      // the species leave our streams before these die
        if (p->sp[s] && p->buf) mphv_internal_unbind_fields(p->sp[s], buf_Ec(p), buf_Bc(p));   // ... and our field buffers
        if (p->sstream[s]) cudaStreamDestroy(p->sstream[s]);
        if (p->ev_mom[s]) cudaEventDestroy(p->ev_mom[s]);
    }
    if (p->ev_fields) cudaEventDestroy(p->ev_fields);
    if (p->buf) cudaFree(p->buf);
    cudaGetLastError();
    delete p;
    return MPHV_OK;
}

int mphv_plasma_invalidate_moments(mphv_plasma *p)
{
    if (!p) return MPHV_ERR_ARG;
    p->have_moments = false;            // the next mphv_plasma_step starts with a moments pass over every species
    return MPHV_OK;
}

int mphv_plasma_set_concurrent(mphv_plasma *p, int concurrent)
{
    if (!p) return MPHV_ERR_ARG;
    DevGuard2 dg(p->dev);
    FLD_TRY(p, cudaDeviceSynchronize());
    p->concurrent = concurrent ? 1 : 0;
    return MPHV_OK;
}

int mphv_plasma_step(mphv_plasma *p, double dt, int nsteps)
{
    if (!p) return MPHV_ERR_ARG;
    if (!is_fin(dt) || nsteps < 0) return fail(p, MPHV_ERR_ARG, "dt is not finite or nsteps < 0");
    mphv_maxwell *m = p->m;
    if (!m->E || !m->B) return fail(p, MPHV_ERR_STATE, "fields not bound (mphv_maxwell_bind)");
    DevGuard2 dg(p->dev);
    const int S = p->ns_species;
    cudaStream_t fs = m->stream;
    int st;
    auto species_stream = [&](int s) { return p->concurrent ? p->sstream[s] : fs; };
    auto sp_fail = [&](int s, int code) { return fail(p, code, "species %d: %s", s, mphv_last_error(p->sp[s])); };
    for (int s = 0; s < S; ++s)
        if ((st = mphv_set_stream(p->sp[s], species_stream(s))) != MPHV_OK) return sp_fail(s, st);
    // everything enqueued on the field stream so far (initial data, earlier calls) precedes the species' work
    FLD_TRY(p, cudaEventRecord(p->ev_fields, fs));
    for (int s = 0; s < S; ++s) {
        if (p->concurrent) FLD_TRY(p, cudaStreamWaitEvent(p->sstream[s], p->ev_fields, 0));
        if (!p->have_moments) {
            double *n = mom_n(p, s);
            if ((st = mphv_moments(p->sp[s], n, n + p->ns, n + 4 * p->ns)) != MPHV_OK) return sp_fail(s, st);
        }
        if (p->concurrent) FLD_TRY(p, cudaEventRecord(p->ev_mom[s], p->sstream[s]));
    }
    p->have_moments = true;

    MaxwellArgs a = base_args(m);
    a.nspecies = S; a.Jout = buf_J(p);
    for (int s = 0; s < S; ++s) { a.q[s] = p->q[s]; a.j[s] = mom_n(p, s) + p->ns; }
    a.dt = 0.5 * dt;
    for (int k = 0; k < nsteps; ++k) {
        // fields: J from the species' present moments, Maxwell(dt/2; J) (after the first step: the closing half
        // step of the previous one and the opening half step of this one, same J), centred fields
        if (p->concurrent)
            for (int s = 0; s < S; ++s) FLD_TRY(p, cudaStreamWaitEvent(fs, p->ev_mom[s], 0));
        a.reps = k == 0 ? 1 : 2;
        a.Ec = buf_Ec(p); a.Bc = buf_Bc(p);
        if ((st = maxwell_run(m, a)) != MPHV_OK) return fail(p, st, "%s", m->err);
        FLD_TRY(p, cudaEventRecord(p->ev_fields, fs));
        // species: frozen centred fields, full split step, moments of the new f
        for (int s = 0; s < S; ++s) {
            if (p->concurrent) FLD_TRY(p, cudaStreamWaitEvent(p->sstream[s], p->ev_fields, 0));
            if ((st = mphv_set_fields_deferred(p->sp[s], buf_Ec(p), buf_Bc(p))) != MPHV_OK) return sp_fail(s, st);
            double *n = mom_n(p, s);
            if ((st = mphv_step_moments(p->sp[s], dt, n, n + p->ns, n + 4 * p->ns)) != MPHV_OK) return sp_fail(s, st);
            if (p->concurrent) FLD_TRY(p, cudaEventRecord(p->ev_mom[s], p->sstream[s]));
        }
    }
    if (nsteps > 0) {                                   // closing half step of the last step
        if (p->concurrent)
            for (int s = 0; s < S; ++s) FLD_TRY(p, cudaStreamWaitEvent(fs, p->ev_mom[s], 0));
        a.reps = 1; a.Ec = nullptr; a.Bc = nullptr;
        if ((st = maxwell_run(m, a)) != MPHV_OK) return fail(p, st, "%s", m->err);
    } else if (p->concurrent) {
        for (int s = 0; s < S; ++s) FLD_TRY(p, cudaStreamWaitEvent(fs, p->ev_mom[s], 0));
    }
    return MPHV_OK;
}

int mphv_plasma_sync(mphv_plasma *p)
{
    if (!p) return MPHV_ERR_ARG;
    DevGuard2 dg(p->dev);
    FLD_TRY(p, cudaStreamSynchronize(p->m->stream));
    for (int s = 0; s < p->ns_species; ++s) {
        int st = mphv_deferred_status(p->sp[s]);
        if (st != MPHV_OK) return fail(p, st, "species %d: %s", s, mphv_last_error(p->sp[s]));
    }
    return MPHV_OK;
}

int mphv_plasma_moments(mphv_plasma *p, int s, double **n, double **j, double **P)
{
    if (!p) return MPHV_ERR_ARG;
    if (s < 0 || s >= p->ns_species) return fail(p, MPHV_ERR_ARG, "species index %d out of range", s);
    if (n) *n = mom_n(p, s);
    if (j) *j = mom_n(p, s) + p->ns;
    if (P) *P = mom_n(p, s) + 4 * p->ns;
    return MPHV_OK;
}

int mphv_plasma_centred_fields(mphv_plasma *p, double **Ec, double **Bc)
{
    if (!p) return MPHV_ERR_ARG;
    if (Ec) *Ec = buf_Ec(p);
    if (Bc) *Bc = buf_Bc(p);
    return MPHV_OK;
}

const char *mphv_plasma_last_error(const mphv_plasma *p) { return p ? p->err : mphv_last_error(nullptr); }

}  // extern "C"
