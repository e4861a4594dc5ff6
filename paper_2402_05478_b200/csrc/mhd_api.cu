// mhd_api.cu — the C ABI of include/mhd.h: context, workspace layout, transform orchestration,
// time stepping, diagnostics.  Host code only enqueues work on the caller's stream; every step of
// the path runs in the kernels of fft_kernels.cu / mhd_kernels.cu.
#include "../../include/mhd.h"
#include "mhd_internal.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

using namespace mhd;

namespace {

constexpr int kMaxShell = 2048;

// kernel classes timed by mhd_profile_begin / mhd_profile_end, in hot-path order
enum { K_Z_INV = 0, K_Y_INV, K_X_C2R, K_PRODUCTS, K_X_R2C, K_XFUSED, K_Y_FWD, K_Z_FWD, K_STAGE, K_NCLASS };
const char* const kClassNames[K_NCLASS] = {"fft_z_inv", "fft_y_inv", "fft_x_c2r", "products", "fft_x_r2c", "x_fused", "fft_y_fwd", "fft_z_fwd", "stage"};

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Geometry {
    int nx, ny, nz;
    int nkx, nky, nkz, px;
    long long npts;       // nx*ny*nz
    long long fieldc;     // complex per compact spectral field  = nkz*nky*px
    long long w1field;    // complex per field after the z inverse = nz*nky*px
    long long w2field;    // complex per field after the y inverse = nz*ny*px
};

bool make_geometry(int nx, int ny, int nz, unsigned flags, Geometry* g) {
    if (!fft_size_supported(nx) || !fft_size_supported(ny)) return false;
    if (nz != 1 && !fft_size_supported(nz)) return false;
    g->nx = nx; g->ny = ny; g->nz = nz;
    if (flags & MHD_FLAG_NO_DEALIAS) {
        g->nkx = nx / 2 + 1; g->nky = ny; g->nkz = nz;
    } else {   // 2/3 rule per axis: keep |k| <= kmax with 3*kmax < n
        g->nkx = (nx - 1) / 3 + 1; g->nky = 2 * ((ny - 1) / 3) + 1; g->nkz = 2 * ((nz - 1) / 3) + 1;
    }
    g->px = (g->nkx + 7) / 8 * 8;
    g->npts = (long long)nx * ny * nz;
    g->fieldc = (long long)g->nkz * g->nky * g->px;
    g->w1field = (long long)nz * g->nky * g->px;
    g->w2field = (long long)nz * ny * g->px;
    return true;
}

struct Layout {
    size_t twx, twy, twz, S, H, Acc, Fh, G, W1, W2, Rf, Rg, red, total;
};

// the fused x pass keeps real-space data in registers: real arrays are then only staging for set/get/diagnostics/forcing
bool use_xfuse(int nx, unsigned flags) { return xfused_supported(nx) && !(flags & MHD_FLAG_UNFUSED_X); }

Layout make_layout(const Geometry& g, int integrator, unsigned flags) {
    Layout L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
    L.twx = take(sizeof(double2) * g.nx);
    L.twy = take(sizeof(double2) * g.ny);
    L.twz = take(sizeof(double2) * g.nz);
    L.S = take(sizeof(double2) * g.fieldc * NFIELD);
    L.H = take(sizeof(double2) * g.fieldc * NFIELD);
    L.Acc = take(integrator == MHD_RK4 ? sizeof(double2) * g.fieldc * NFIELD : 0);
    L.Fh = take((flags & MHD_FLAG_FORCING) ? sizeof(double2) * g.fieldc * 3 : 0);
    L.G = take(sizeof(double2) * g.fieldc * NPROD);
    L.W1 = take(g.nz > 1 ? sizeof(double2) * g.w1field * NPROD : 0);
    L.W2 = take(sizeof(double2) * g.w2field * NPROD);
    L.Rf = take(sizeof(double) * g.npts * NFIELD);
    L.Rg = take(sizeof(double) * g.npts * (use_xfuse(g.nx, flags) ? (int)NFIELD : (int)NPROD));
    L.red = take(sizeof(double) * ((RED_NSUM + 1) * RED_BLOCKS + 64 + 2 * kMaxShell));
    L.total = o;
    return L;
}

void host_twiddles(int n, std::vector<double2>& t) {
    t.resize(n);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int j = 0; j < n; ++j) {
        long double a = two_pi * (long double)j / (long double)n;
        t[j] = make_double2((double)cosl(a), -(double)sinl(a));   // exp(-2 pi i j / n)
    }
}

}  // namespace

struct mhd_ctx {
    Geometry g;
    double nu, eta, cs, dt;
    int integrator;
    unsigned flags;
    int hydro;
    cudaStream_t st;
    int device;                // the device that owns the workspace: every call runs with it current (DeviceGuard)
    char* ws;
    Layout L;
    double2 *twx, *twy, *twz, *S, *H, *Acc, *Fh, *G, *W1, *W2;
    double kf[3];              // 2*pi/L per axis (1.0 on the 2*pi box)
    int have_forcing;          // Fh holds a force (mhd_set_forcing)
    double *Rf, *Rg, *red_partial, *red_result, *spec_dev;
    long long step;
    int have_fields, have_history;
    cudaGraphExec_t graph;     // one steady-state step (AB2 non-first / RK4), replayed by mhd_step
    int graph_ready;
    long long graph_launches;  // kernels inside the captured step
    int xfuse;                 // fused x pass available for this nx (and not disabled by MHD_FLAG_UNFUSED_X)
    int profiling;             // mhd_profile_begin: eager steps with CUDA events around every kernel
    std::vector<cudaEvent_t>* prof_ev;   // [K_NCLASS] start/stop pairs
    char err[256];
};

namespace {

// Makes `device` current for the duration of one API call and restores the caller's device afterwards, so a context
// (or plan) created on one GPU can be driven while another GPU is current.
// device < 0 (owner unknown) leaves the caller's device in place by design; a device that is known but cannot be made
// current sets `failed`, and the API call returns MHD_ECUDA instead of running on the wrong GPU.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    bool failed = false;
    explicit DeviceGuard(int device) {
        if (device < 0) return;
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); failed = true; return; }
        if (prev == device) return;
        if (cudaSetDevice(device) == cudaSuccess) switched = true;
        else { cudaGetLastError(); failed = true; }
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};
// a stream created on another GPU than the workspace's cannot carry this context's work (false only when that is certain)
bool stream_on_device(cudaStream_t st, int device) {
    if (!st || device < 0) return true;          // legacy default stream: belongs to whichever device is current
    int sd = -1;
    if (cudaStreamGetDevice(st, &sd) != cudaSuccess) { cudaGetLastError(); return true; }
    return sd == device;
}
const char* const kGuardFailed = "cannot make the GPU that owns the workspace current";
// device that owns a device pointer (-1 if it cannot be determined: the current device is then used as is)
int owning_device(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return -1; }
    return (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) ? at.device : -1;
}

int fail(mhd_ctx* c, int code, const char* what, cudaError_t e = cudaSuccess) {
    if (c) {
        if (e != cudaSuccess) snprintf(c->err, sizeof(c->err), "%s: %s", what, cudaGetErrorString(e));
        else snprintf(c->err, sizeof(c->err), "%s", what);
    }
    return code;
}
#define CK(call)                                                        \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return fail(c, MHD_ECUDA, #call, e_);    \
    } while (0)

// run `launch` (one kernel) and, when profiling, bracket it with CUDA events on the context's stream
template <typename F>
cudaError_t timed(mhd_ctx* c, int cls, F launch) {
    if (!c->profiling) return launch();
    cudaEvent_t a, b;
    cudaError_t e;
    if ((e = cudaEventCreate(&a)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&b)) != cudaSuccess) { cudaEventDestroy(a); return e; }
    cudaEventRecord(a, c->st);
    e = launch();
    cudaEventRecord(b, c->st);
    c->prof_ev[cls].push_back(a);
    c->prof_ev[cls].push_back(b);
    return e;
}

SpecGeom spec_geom(const Geometry& g) {
    SpecGeom s;
    s.nx = g.nx; s.ny = g.ny; s.nz = g.nz; s.nkx = g.nkx; s.nky = g.nky; s.nkz = g.nkz; s.px = g.px; s.field = g.fieldc;
    return s;
}

// compact spectral fields -> W2 = [field][z][y][px] half-spectrum rows (z inverse, y inverse)
cudaError_t inverse_zy(mhd_ctx* c, const double2* src, int nf) {
    const Geometry& g = c->g;
    cudaError_t e;
    const double2* ysrc = src;
    long long ysrc_outer = (long long)g.nky * g.px;   // per (field, z) slab; with nz == 1 this is the field stride
    if (g.nz > 1) {
        AxisArgs a;
        a.in = src; a.out = c->W1; a.nouter = nf;
        a.in_outer = g.fieldc; a.out_outer = g.w1field;
        a.in_row = a.out_row = (long long)g.nky * g.px;
        a.inner = g.nky * g.px; a.nk_in = g.nkz; a.nk_out = g.nz; a.scale = 1.0;
        if ((e = timed(c, K_Z_INV, [&] { return launch_fft_axis(g.nz, true, a, c->twz, c->st); })) != cudaSuccess) return e;
        ysrc = c->W1;
    }
    {
        AxisArgs a;
        a.in = ysrc; a.out = c->W2; a.nouter = (long long)nf * g.nz;
        a.in_outer = ysrc_outer; a.out_outer = (long long)g.ny * g.px;
        a.in_row = a.out_row = g.px;
        a.inner = g.px; a.nk_in = g.nky; a.nk_out = g.ny; a.scale = 1.0;
        if ((e = timed(c, K_Y_INV, [&] { return launch_fft_axis(g.ny, true, a, c->twy, c->st); })) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// compact spectral fields -> real fields  (z inverse, y inverse, x complex-to-real)
cudaError_t inverse_fields(mhd_ctx* c, const double2* src, int nf, double* real_out) {
    const Geometry& g = c->g;
    cudaError_t e;
    if ((e = inverse_zy(c, src, nf)) != cudaSuccess) return e;
    RowArgs r;
    r.spec = c->W2; r.real = real_out; r.spec_pitch = g.px; r.real_pitch = g.nx;
    r.nrows = (long long)nf * g.nz * g.ny; r.nkx = g.nkx; r.scale = 1.0 / (double)g.npts;
    return timed(c, K_X_C2R, [&] { return launch_fft_rows(g.nx, true, r, c->twx, c->st); });
}

cudaError_t forward_yz(mhd_ctx* c, int nf, double2* dst);

// real fields -> compact spectral fields (x real-to-complex, y forward, z forward), unnormalised
cudaError_t forward_fields(mhd_ctx* c, const double* real_in, int nf, double2* dst) {
    const Geometry& g = c->g;
    cudaError_t e;
    RowArgs r;
    r.spec = c->W2; r.real = const_cast<double*>(real_in); r.spec_pitch = g.px; r.real_pitch = g.nx;
    r.nrows = (long long)nf * g.nz * g.ny; r.nkx = g.nkx; r.scale = 1.0;
    if ((e = timed(c, K_X_R2C, [&] { return launch_fft_rows(g.nx, false, r, c->twx, c->st); })) != cudaSuccess) return e;
    return forward_yz(c, nf, dst);
}

// W2 half-spectrum rows -> compact spectral fields (y forward, z forward)
cudaError_t forward_yz(mhd_ctx* c, int nf, double2* dst) {
    const Geometry& g = c->g;
    cudaError_t e;
    {
        AxisArgs a;
        a.in = c->W2; a.out = (g.nz > 1) ? c->W1 : dst; a.nouter = (long long)nf * g.nz;
        a.in_outer = (long long)g.ny * g.px; a.out_outer = (long long)g.nky * g.px;
        a.in_row = a.out_row = g.px;
        a.inner = g.px; a.nk_in = g.ny; a.nk_out = g.nky; a.scale = 1.0;
        if ((e = timed(c, K_Y_FWD, [&] { return launch_fft_axis(g.ny, false, a, c->twy, c->st); })) != cudaSuccess) return e;
    }
    if (g.nz > 1) {
        AxisArgs a;
        a.in = c->W1; a.out = dst; a.nouter = nf;
        a.in_outer = g.w1field; a.out_outer = g.fieldc;
        a.in_row = a.out_row = (long long)g.nky * g.px;
        a.inner = g.nky * g.px; a.nk_in = g.nz; a.nk_out = g.nkz; a.scale = 1.0;
        if ((e = timed(c, K_Z_FWD, [&] { return launch_fft_axis(g.nz, false, a, c->twz, c->st); })) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// one right-hand-side evaluation followed by the integrator stage `mode`
cudaError_t rhs_stage(mhd_ctx* c, int mode) {
    const Geometry& g = c->g;
    cudaError_t e;
    if (c->xfuse) {   // x inverse + products + x forward in one kernel, in place on W2
        if ((e = inverse_zy(c, c->S, c->hydro ? 4 : NFIELD)) != cudaSuccess) return e;
        XFusedArgs x;
        x.w2 = c->W2; x.field_stride = g.w2field; x.nrows = (long long)g.nz * g.ny; x.px = g.px; x.nkx = g.nkx;
        x.scale = 1.0 / (double)g.npts;
        if ((e = timed(c, K_XFUSED, [&] { return launch_xfused(g.nx, x, c->hydro, c->twx, c->st); })) != cudaSuccess) return e;
        if ((e = forward_yz(c, c->hydro ? 9 : NPROD, c->G)) != cudaSuccess) return e;
    } else {
        if ((e = inverse_fields(c, c->S, c->hydro ? 4 : NFIELD, c->Rf)) != cudaSuccess) return e;
        if ((e = timed(c, K_PRODUCTS, [&] { return launch_products(c->Rf, c->Rg, g.npts, c->hydro, c->st); })) != cudaSuccess) return e;
        if ((e = forward_fields(c, c->Rg, c->hydro ? 9 : NPROD, c->G)) != cudaSuccess) return e;
    }
    StageArgs s;
    s.g = spec_geom(g); s.S = c->S; s.G = c->G; s.H = c->H; s.Acc = c->Acc;
    s.nu = c->nu; s.eta = c->eta; s.cs2 = c->cs * c->cs; s.dt = c->dt; s.mode = mode; s.hydro = c->hydro;
    s.F = c->have_forcing ? c->Fh : nullptr; s.kfx = c->kf[0]; s.kfy = c->kf[1]; s.kfz = c->kf[2];
    return timed(c, K_STAGE, [&] { return launch_stage(s, c->st); });
}

cudaError_t one_step(mhd_ctx* c, bool first_ab2) {
    cudaError_t e;
    if (c->integrator == MHD_AB2) return rhs_stage(c, first_ab2 ? STAGE_AB2_EULER : STAGE_AB2);
    for (int s = STAGE_RK4_1; s <= STAGE_RK4_4; ++s)
        if ((e = rhs_stage(c, s)) != cudaSuccess) return e;
    return cudaSuccess;
}

}  // namespace

// ================================================================================================
// C ABI
// ================================================================================================
extern "C" {

const char* mhd_strerror(int code) {
    switch (code) {
        case MHD_OK: return "ok";
        case MHD_EINVAL: return "invalid argument";
        case MHD_ENOMEM: return "out of host memory";
        case MHD_ECUDA: return "CUDA error";
        case MHD_ESTATE: return "call out of order (no fields set)";
        case MHD_ENONFINITE: return "non-finite value or non-positive density in the state";
        default: return "unknown error code";
    }
}

const char* mhd_last_error(const mhd_ctx* c) { return c ? c->err : ""; }

long long mhd_launch_count(void) { return launch_count(); }

int mhd_profile_kernel_count(void) { return K_NCLASS; }
const char* mhd_profile_kernel_name(int i) { return (i >= 0 && i < K_NCLASS) ? kClassNames[i] : ""; }

int mhd_measure_peaks(void* scratch, size_t bytes, void* stream, double* fp64_tflops, double* smem_gbs) {
    if (!scratch || !fp64_tflops || !smem_gbs || bytes < ((size_t)4 << 20)) return MHD_EINVAL;
    DeviceGuard guard(owning_device(scratch));
    if (guard.failed) return MHD_ECUDA;
    return measure_peaks((double*)scratch, bytes / sizeof(double), (cudaStream_t)stream, fp64_tflops, smem_gbs) == cudaSuccess ? MHD_OK : MHD_ECUDA;
}

int mhd_measure_exchange(void* scratch, size_t bytes, void* stream, int dfma_per_exchange, int barrier_mode, double* smem_gbs) {
    if (!scratch || !smem_gbs || bytes < ((size_t)4 << 20)) return MHD_EINVAL;
    if (dfma_per_exchange < 0 || dfma_per_exchange > 256 || dfma_per_exchange % 64 != 0) return MHD_EINVAL;
    if (barrier_mode < 0 || barrier_mode > 3) return MHD_EINVAL;
    DeviceGuard guard(owning_device(scratch));
    if (guard.failed) return MHD_ECUDA;
    return measure_exchange((double*)scratch, bytes / sizeof(double), (cudaStream_t)stream, dfma_per_exchange, barrier_mode, smem_gbs) == cudaSuccess ? MHD_OK : MHD_ECUDA;
}

int mhd_profile_begin(mhd_ctx* c) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    for (int k = 0; k < K_NCLASS; ++k) {
        for (cudaEvent_t ev : c->prof_ev[k]) cudaEventDestroy(ev);
        c->prof_ev[k].clear();
    }
    c->profiling = 1;
    return MHD_OK;
}

int mhd_profile_end(mhd_ctx* c, int* counts, double* ms) {
    if (!c || !counts || !ms) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    c->profiling = 0;
    CK(cudaStreamSynchronize(c->st));
    for (int k = 0; k < K_NCLASS; ++k) {
        counts[k] = (int)(c->prof_ev[k].size() / 2);
        double tot = 0.0;
        for (size_t i = 0; i + 1 < c->prof_ev[k].size(); i += 2) {
            float t = 0.f;
            CK(cudaEventElapsedTime(&t, c->prof_ev[k][i], c->prof_ev[k][i + 1]));
            tot += t;
        }
        ms[k] = tot;
        for (cudaEvent_t ev : c->prof_ev[k]) cudaEventDestroy(ev);
        c->prof_ev[k].clear();
    }
    return MHD_OK;
}

size_t mhd_workspace_bytes(int nx, int ny, int nz, int integrator, unsigned flags) {
    Geometry g;
    if (!make_geometry(nx, ny, nz, flags, &g)) return 0;
    if (integrator != MHD_AB2 && integrator != MHD_RK4) return 0;
    return make_layout(g, integrator, flags).total;
}

int mhd_create(mhd_ctx** out, int nx, int ny, int nz, double nu, double eta, double cs, double dt,
               int integrator, unsigned flags, void* workspace, size_t workspace_bytes, void* stream) {
    if (!out) return MHD_EINVAL;
    *out = nullptr;
    Geometry g;
    if (!make_geometry(nx, ny, nz, flags, &g)) return MHD_EINVAL;
    if (integrator != MHD_AB2 && integrator != MHD_RK4) return MHD_EINVAL;
    if (!(nu >= 0.0) || !(eta >= 0.0) || !(cs >= 0.0) || !(dt > 0.0)) return MHD_EINVAL;
    if (!isfinite(nu) || !isfinite(eta) || !isfinite(cs) || !isfinite(dt)) return MHD_EINVAL;
    if (flags & ~(MHD_FLAG_HYDRO | MHD_FLAG_NO_DEALIAS | MHD_FLAG_FORCING | MHD_FLAG_UNFUSED_X | MHD_FLAG_NO_GRAPH))
        return MHD_EINVAL;
    const Layout L = make_layout(g, integrator, flags);
    if (!workspace || workspace_bytes < L.total || ((size_t)workspace & 255u)) return MHD_EINVAL;
    mhd_ctx* c = new (std::nothrow) mhd_ctx();
    if (!c) return MHD_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->g = g; c->nu = nu; c->eta = eta; c->cs = cs; c->dt = dt;
    c->integrator = integrator; c->flags = flags; c->hydro = (flags & MHD_FLAG_HYDRO) ? 1 : 0;
    c->st = (cudaStream_t)stream; c->ws = (char*)workspace; c->L = L;
    c->device = owning_device(workspace);
    DeviceGuard guard(c->device);
    if (guard.failed) { delete c; return MHD_ECUDA; }
    if (!stream_on_device((cudaStream_t)stream, c->device)) { delete c; return MHD_EINVAL; }
    c->xfuse = use_xfuse(nx, flags);
    c->prof_ev = new (std::nothrow) std::vector<cudaEvent_t>[K_NCLASS];
    if (!c->prof_ev) { delete c; return MHD_ENOMEM; }
    c->twx = (double2*)(c->ws + L.twx); c->twy = (double2*)(c->ws + L.twy); c->twz = (double2*)(c->ws + L.twz);
    c->S = (double2*)(c->ws + L.S); c->H = (double2*)(c->ws + L.H); c->Acc = (double2*)(c->ws + L.Acc);
    c->Fh = (double2*)(c->ws + L.Fh); c->kf[0] = c->kf[1] = c->kf[2] = 1.0;
    c->G = (double2*)(c->ws + L.G); c->W1 = (double2*)(c->ws + L.W1); c->W2 = (double2*)(c->ws + L.W2);
    c->Rf = (double*)(c->ws + L.Rf); c->Rg = (double*)(c->ws + L.Rg);
    c->red_partial = (double*)(c->ws + L.red);
    c->red_result = c->red_partial + (RED_NSUM + 1) * RED_BLOCKS;
    c->spec_dev = c->red_result + 64;
    // zero everything once: pad columns and unused fields are then never anything but zero
    cudaError_t e = cudaMemsetAsync(c->ws, 0, L.total, c->st);
    std::vector<double2> t;
    const int n3[3] = {nx, ny, nz};
    double2* d3[3] = {c->twx, c->twy, c->twz};
    for (int a = 0; a < 3 && e == cudaSuccess; ++a) {
        host_twiddles(n3[a], t);
        e = cudaMemcpyAsync(d3[a], t.data(), sizeof(double2) * n3[a], cudaMemcpyHostToDevice, c->st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);   // t is reused / freed
    }
    if (e != cudaSuccess) { delete[] c->prof_ev; delete c; return MHD_ECUDA; }
    *out = c;
    return MHD_OK;
}

void mhd_destroy(mhd_ctx* c) {
    if (!c) return;
    DeviceGuard guard(c->device);
    if (c->graph) cudaGraphExecDestroy(c->graph);
    if (c->prof_ev) {
        for (int k = 0; k < K_NCLASS; ++k) for (cudaEvent_t ev : c->prof_ev[k]) cudaEventDestroy(ev);
        delete[] c->prof_ev;
    }
    delete c;
}

// the captured step bakes in the stage kernel's arguments: drop it when they change
static void invalidate_graph(mhd_ctx* c) {
    if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
    c->graph_ready = 0;
}

int mhd_set_box(mhd_ctx* c, double lx, double ly, double lz) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0) || !isfinite(lx) || !isfinite(ly) || !isfinite(lz))
        return fail(c, MHD_EINVAL, "mhd_set_box: lengths must be finite and > 0");
    const double two_pi = 6.283185307179586476925286766559;
    const double l[3] = {lx, ly, lz};
    for (int i = 0; i < 3; ++i) c->kf[i] = (l[i] == two_pi) ? 1.0 : two_pi / l[i];
    invalidate_graph(c);
    return MHD_OK;
}

int mhd_set_forcing(mhd_ctx* c, const double* fx, const double* fy, const double* fz) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!fx && !fy && !fz) { c->have_forcing = 0; invalidate_graph(c); return MHD_OK; }
    if (!fx || !fy || !fz) return fail(c, MHD_EINVAL, "mhd_set_forcing: give all three components or none");
    if (!(c->flags & MHD_FLAG_FORCING)) return fail(c, MHD_ESTATE, "mhd_set_forcing: context created without MHD_FLAG_FORCING");
    const long long n = c->g.npts;
    const size_t fb = sizeof(double) * n;
    const double* f[3] = {fx, fy, fz};
    for (int i = 0; i < 3; ++i)
        if (f[i] != c->Rg + i * n) CK(cudaMemcpyAsync(c->Rg + i * n, f[i], fb, cudaMemcpyDeviceToDevice, c->st));
    CK(forward_fields(c, c->Rg, 3, c->Fh));
    c->have_forcing = 1;
    invalidate_graph(c);
    return MHD_OK;
}

int mhd_set_forcing_host(mhd_ctx* c, const double* fx, const double* fy, const double* fz) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!fx && !fy && !fz) return mhd_set_forcing(c, nullptr, nullptr, nullptr);
    if (!fx || !fy || !fz) return fail(c, MHD_EINVAL, "mhd_set_forcing_host: give all three components or none");
    if (!(c->flags & MHD_FLAG_FORCING)) return fail(c, MHD_ESTATE, "mhd_set_forcing_host: context created without MHD_FLAG_FORCING");
    const long long n = c->g.npts;
    const double* f[3] = {fx, fy, fz};
    for (int i = 0; i < 3; ++i) CK(cudaMemcpyAsync(c->Rg + i * n, f[i], sizeof(double) * n, cudaMemcpyHostToDevice, c->st));
    return mhd_set_forcing(c, c->Rg, c->Rg + n, c->Rg + 2 * n);
}

int mhd_set_fields(mhd_ctx* c, const double* rho, const double* ux, const double* uy, const double* uz,
                   const double* bx, const double* by, const double* bz) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!rho || !ux || !uy || !uz) return fail(c, MHD_EINVAL, "mhd_set_fields: NULL field");
    if (!c->hydro && (!bx || !by || !bz)) return fail(c, MHD_EINVAL, "mhd_set_fields: NULL magnetic field without MHD_FLAG_HYDRO");
    const long long n = c->g.npts;
    const size_t fb = sizeof(double) * n;
    CK(cudaMemcpyAsync(c->Rf + F_RHO * n, rho, fb, cudaMemcpyDeviceToDevice, c->st));
    CK(launch_momentum(rho, ux, uy, uz, c->Rf + F_MX * n, n, c->st));
    if (!c->hydro) {
        CK(cudaMemcpyAsync(c->Rf + F_BX * n, bx, fb, cudaMemcpyDeviceToDevice, c->st));
        CK(cudaMemcpyAsync(c->Rf + F_BY * n, by, fb, cudaMemcpyDeviceToDevice, c->st));
        CK(cudaMemcpyAsync(c->Rf + F_BZ * n, bz, fb, cudaMemcpyDeviceToDevice, c->st));
    }
    CK(forward_fields(c, c->Rf, c->hydro ? 4 : NFIELD, c->S));
    c->have_fields = 1; c->have_history = 0; c->step = 0;
    return MHD_OK;
}

int mhd_set_fields_host(mhd_ctx* c, const double* rho, const double* ux, const double* uy, const double* uz,
                        const double* bx, const double* by, const double* bz) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!rho || !ux || !uy || !uz) return fail(c, MHD_EINVAL, "mhd_set_fields_host: NULL field");
    if (!c->hydro && (!bx || !by || !bz)) return fail(c, MHD_EINVAL, "mhd_set_fields_host: NULL magnetic field");
    const long long n = c->g.npts;
    const size_t fb = sizeof(double) * n;
    const double* h[7] = {rho, ux, uy, uz, bx, by, bz};
    const int nf = c->hydro ? 4 : 7;
    for (int i = 0; i < nf; ++i) CK(cudaMemcpyAsync(c->Rg + i * n, h[i], fb, cudaMemcpyHostToDevice, c->st));
    double* d = c->Rg;
    return mhd_set_fields(c, d, d + n, d + 2 * n, d + 3 * n, c->hydro ? nullptr : d + 4 * n,
                          c->hydro ? nullptr : d + 5 * n, c->hydro ? nullptr : d + 6 * n);
}

int mhd_step(mhd_ctx* c, int nsteps) {
    if (!c || nsteps < 0) return c ? fail(c, MHD_EINVAL, "mhd_step: nsteps < 0") : MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!c->have_fields) return fail(c, MHD_ESTATE, "mhd_step before mhd_set_fields");
    int done = 0;
    // a launch failure part-way through still leaves `done` completed steps in the state: account for them
#define CKS(call)                                                                         \
    do {                                                                                  \
        cudaError_t e_ = (call);                                                          \
        if (e_ != cudaSuccess) { c->step += done; return fail(c, MHD_ECUDA, #call, e_); } \
    } while (0)
    if (nsteps > 0 && c->integrator == MHD_AB2 && !c->have_history) {
        CKS(one_step(c, true));
        c->have_history = 1;
        done = 1;
    }
    const bool no_graph = (c->flags & MHD_FLAG_NO_GRAPH) != 0;
    while (done < nsteps) {
        const int left = nsteps - done;
        if (!no_graph && !c->profiling && c->st != nullptr && (c->graph_ready || left >= 3)) {
            if (!c->graph_ready) {
                CKS(one_step(c, false));   // eager once: sets kernel attributes outside capture
                ++done;
                const long long before = launch_count();
                cudaGraph_t gr = nullptr;
                CKS(cudaStreamBeginCapture(c->st, cudaStreamCaptureModeThreadLocal));
                cudaError_t e = one_step(c, false);
                cudaError_t e2 = cudaStreamEndCapture(c->st, &gr);
                if (e != cudaSuccess || e2 != cudaSuccess) {
                    if (gr) cudaGraphDestroy(gr);
                    c->step += done;
                    return fail(c, MHD_ECUDA, "graph capture", e != cudaSuccess ? e : e2);
                }
                c->graph_launches = launch_count() - before;
                add_launches(-c->graph_launches);   // capture enqueued nothing
                e = cudaGraphInstantiate(&c->graph, gr, 0);
                cudaGraphDestroy(gr);
                if (e != cudaSuccess) { c->step += done; return fail(c, MHD_ECUDA, "cudaGraphInstantiate", e); }
                c->graph_ready = 1;
                continue;
            }
            CKS(cudaGraphLaunch(c->graph, c->st));
            add_launches(c->graph_launches);
            ++done;
        } else {
            CKS(one_step(c, false));
            ++done;
        }
    }
#undef CKS
    c->step += nsteps;
    return MHD_OK;
}

int mhd_get_fields(mhd_ctx* c, double* rho, double* ux, double* uy, double* uz, double* bx, double* by, double* bz) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!rho || !ux || !uy || !uz) return fail(c, MHD_EINVAL, "mhd_get_fields: NULL field");
    if (!c->have_fields) return fail(c, MHD_ESTATE, "mhd_get_fields before mhd_set_fields");
    const long long n = c->g.npts;
    const size_t fb = sizeof(double) * n;
    CK(inverse_fields(c, c->S, c->hydro ? 4 : NFIELD, c->Rf));
    CK(cudaMemcpyAsync(rho, c->Rf + F_RHO * n, fb, cudaMemcpyDeviceToDevice, c->st));
    CK(launch_velocity(c->Rf, ux, uy, uz, n, c->st));
    double* b[3] = {bx, by, bz};
    for (int i = 0; i < 3; ++i) {
        if (!b[i]) continue;
        if (c->hydro) CK(cudaMemsetAsync(b[i], 0, fb, c->st));
        else CK(cudaMemcpyAsync(b[i], c->Rf + (F_BX + i) * n, fb, cudaMemcpyDeviceToDevice, c->st));
    }
    return MHD_OK;
}

int mhd_get_fields_host(mhd_ctx* c, double* rho, double* ux, double* uy, double* uz, double* bx, double* by, double* bz) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!rho || !ux || !uy || !uz) return fail(c, MHD_EINVAL, "mhd_get_fields_host: NULL field");
    if (!c->have_fields) return fail(c, MHD_ESTATE, "mhd_get_fields_host before mhd_set_fields");
    const long long n = c->g.npts;
    const size_t fb = sizeof(double) * n;
    CK(inverse_fields(c, c->S, c->hydro ? 4 : NFIELD, c->Rf));
    CK(launch_velocity3(c->Rf, c->Rg, n, c->st));
    CK(cudaMemcpyAsync(rho, c->Rf + F_RHO * n, fb, cudaMemcpyDeviceToHost, c->st));
    double* u[3] = {ux, uy, uz};
    double* b[3] = {bx, by, bz};
    for (int i = 0; i < 3; ++i) CK(cudaMemcpyAsync(u[i], c->Rg + i * n, fb, cudaMemcpyDeviceToHost, c->st));
    for (int i = 0; i < 3; ++i) {
        if (!b[i]) continue;
        if (c->hydro) memset(b[i], 0, fb);
        else CK(cudaMemcpyAsync(b[i], c->Rf + (F_BX + i) * n, fb, cudaMemcpyDeviceToHost, c->st));
    }
    CK(cudaStreamSynchronize(c->st));
    return MHD_OK;
}

namespace {
struct StateHeader {          // first 256 bytes of the blob
    unsigned long long magic;
    int nx, ny, nz, integrator;
    unsigned flags;
    int have_fields, have_history;
    long long step;
};
constexpr unsigned long long kStateMagic = 0x4d48443153544154ull;   // "MHD1STAT"
constexpr size_t kStateHeaderBytes = 256;
}  // namespace

size_t mhd_state_bytes(const mhd_ctx* c) {
    if (!c) return 0;
    return kStateHeaderBytes + 2 * sizeof(double2) * (size_t)c->g.fieldc * NFIELD;      // header + S + H
}

int mhd_get_state(mhd_ctx* c, void* state, size_t bytes) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!state || bytes < mhd_state_bytes(c)) return fail(c, MHD_EINVAL, "mhd_get_state: buffer missing or too small");
    if (!c->have_fields) return fail(c, MHD_ESTATE, "mhd_get_state before mhd_set_fields");
    StateHeader h;
    memset(&h, 0, sizeof(h));
    h.magic = kStateMagic; h.nx = c->g.nx; h.ny = c->g.ny; h.nz = c->g.nz; h.integrator = c->integrator;
    h.flags = c->flags & (MHD_FLAG_HYDRO | MHD_FLAG_NO_DEALIAS);
    h.have_fields = c->have_fields; h.have_history = c->have_history; h.step = c->step;
    const size_t fb = sizeof(double2) * (size_t)c->g.fieldc * NFIELD;
    char* d = (char*)state;
    CK(cudaMemsetAsync(d, 0, kStateHeaderBytes, c->st));
    CK(cudaMemcpyAsync(d, &h, sizeof(h), cudaMemcpyHostToDevice, c->st));
    CK(cudaStreamSynchronize(c->st));                      // h lives on this stack frame
    CK(cudaMemcpyAsync(d + kStateHeaderBytes, c->S, fb, cudaMemcpyDeviceToDevice, c->st));
    CK(cudaMemcpyAsync(d + kStateHeaderBytes + fb, c->H, fb, cudaMemcpyDeviceToDevice, c->st));
    return MHD_OK;
}

int mhd_set_state(mhd_ctx* c, const void* state, size_t bytes) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!state || bytes < mhd_state_bytes(c)) return fail(c, MHD_EINVAL, "mhd_set_state: buffer missing or too small");
    StateHeader h;
    CK(cudaMemcpyAsync(&h, state, sizeof(h), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    if (h.magic != kStateMagic || h.nx != c->g.nx || h.ny != c->g.ny || h.nz != c->g.nz || h.integrator != c->integrator ||
        h.flags != (c->flags & (MHD_FLAG_HYDRO | MHD_FLAG_NO_DEALIAS)) || !h.have_fields)
        return fail(c, MHD_EINVAL, "mhd_set_state: the blob was written by a different configuration");
    const size_t fb = sizeof(double2) * (size_t)c->g.fieldc * NFIELD;
    const char* d = (const char*)state;
    CK(cudaMemcpyAsync(c->S, d + kStateHeaderBytes, fb, cudaMemcpyDeviceToDevice, c->st));
    CK(cudaMemcpyAsync(c->H, d + kStateHeaderBytes + fb, fb, cudaMemcpyDeviceToDevice, c->st));
    c->have_fields = 1; c->have_history = h.have_history; c->step = h.step;
    return MHD_OK;
}

int mhd_diagnostics(mhd_ctx* c, mhd_diag* out, double* ekin_spec, double* emag_spec, int nshell) {
    if (!c) return MHD_EINVAL;
    DeviceGuard guard(c->device);
    if (guard.failed) return fail(c, MHD_ECUDA, kGuardFailed);
    if (!out || nshell < 0 || nshell > kMaxShell || (nshell > 0 && (!ekin_spec || !emag_spec)))
        return fail(c, MHD_EINVAL, "mhd_diagnostics: bad argument");
    if (!c->have_fields) return fail(c, MHD_ESTATE, "mhd_diagnostics before mhd_set_fields");
    const Geometry& g = c->g;
    const long long n = g.npts;
    const SpecGeom sg = spec_geom(g);
    if (nshell > 0 && (c->kf[0] != 1.0 || c->kf[1] != 1.0 || (g.nz > 1 && c->kf[2] != 1.0)))
        return fail(c, MHD_EINVAL, "mhd_diagnostics: shell spectra are defined on the 2*pi box only");
    CK(inverse_fields(c, c->S, c->hydro ? 4 : NFIELD, c->Rf));
    CK(launch_reduce_fields(c->Rf, n, c->hydro, c->red_partial, c->red_result, c->st));
    {
        // Velocity spectrum and the paper's diagnostics (Omega(t), Rayleigh quotient): u = m/rho is not band-limited, and the spectrum is defined over ALL modes
        // (it sums to 1/2 <|u|^2>), so u^ comes from an unpruned forward transform:
        // x pass into W2 viewed as [3][nz][ny][pxf], then y and z in place.
        CK(launch_velocity3(c->Rf, c->Rg, n, c->st));
        SpecGeom fg;
        fg.nx = g.nx; fg.ny = g.ny; fg.nz = g.nz; fg.nkx = g.nx / 2 + 1; fg.nky = g.ny; fg.nkz = g.nz;
        fg.px = (fg.nkx + 7) / 8 * 8; fg.field = (long long)g.nz * g.ny * fg.px;
        RowArgs r;
        r.spec = c->W2; r.real = c->Rg; r.spec_pitch = fg.px; r.real_pitch = g.nx;
        r.nrows = 3LL * g.nz * g.ny; r.nkx = fg.nkx; r.scale = 1.0;
        CK(launch_fft_rows(g.nx, false, r, c->twx, c->st));
        AxisArgs a;
        a.in = c->W2; a.out = c->W2; a.nouter = 3LL * g.nz; a.in_outer = a.out_outer = (long long)g.ny * fg.px;
        a.in_row = a.out_row = fg.px; a.inner = fg.px; a.nk_in = a.nk_out = g.ny; a.scale = 1.0;
        CK(launch_fft_axis(g.ny, false, a, c->twy, c->st));
        if (g.nz > 1) {
            a.nouter = 3; a.in_outer = a.out_outer = fg.field; a.in_row = a.out_row = (long long)g.ny * fg.px;
            a.inner = g.ny * fg.px; a.nk_in = a.nk_out = g.nz;
            CK(launch_fft_axis(g.nz, false, a, c->twz, c->st));
        }
        CK(launch_reduce_curl(fg, c->W2, c->kf[0], c->kf[1], c->kf[2], c->red_partial, c->red_result + 20, c->st));
        if (c->hydro) CK(cudaMemsetAsync(c->red_result + 24, 0, 2 * sizeof(double), c->st));
        else CK(launch_reduce_curl(sg, c->S + F_BX * g.fieldc, c->kf[0], c->kf[1], c->kf[2], c->red_partial, c->red_result + 24, c->st));
        if (nshell > 0) {
            CK(launch_spectrum(fg, c->W2, (double*)c->G, c->spec_dev, nshell, c->st));
            if (c->hydro) CK(cudaMemsetAsync(c->spec_dev + kMaxShell, 0, sizeof(double) * nshell, c->st));
            else CK(launch_spectrum(sg, c->S + F_BX * g.fieldc, (double*)c->G, c->spec_dev + kMaxShell, nshell, c->st));
        }
    }
    if (!c->hydro) {
        CK(launch_divb_spec(sg, c->S + F_BX * g.fieldc, c->G, c->kf[0], c->kf[1], c->kf[2], c->st));
        CK(inverse_fields(c, c->G, 1, c->Rg));
        CK(launch_reduce_maxabs(c->Rg, n, c->red_partial, c->red_result + 16, c->st));
    } else {
        CK(cudaMemsetAsync(c->red_result + 16, 0, 2 * sizeof(double), c->st));
    }
    double r[32];   // [0..10] field sums + bad flag, [16..17] max|div B| + bad flag, [20..21] curl u / u sums, [24..25] curl B / B sums
    CK(cudaMemcpyAsync(r, c->red_result, sizeof(r), cudaMemcpyDeviceToHost, c->st));
    if (nshell > 0) {
        CK(cudaMemcpyAsync(ekin_spec, c->spec_dev, sizeof(double) * nshell, cudaMemcpyDeviceToHost, c->st));
        CK(cudaMemcpyAsync(emag_spec, c->spec_dev + kMaxShell, sizeof(double) * nshell, cudaMemcpyDeviceToHost, c->st));
    }
    CK(cudaStreamSynchronize(c->st));
    const double inv = 1.0 / (double)n;
    out->step = c->step; out->time = (double)c->step * c->dt;
    out->ekin = r[0] * inv; out->emag = r[1] * inv; out->eiso = c->cs * c->cs * r[2] * inv; out->mass = r[3] * inv;
    for (int i = 0; i < 3; ++i) { out->mom[i] = r[4 + i] * inv; out->bmean[i] = r[7 + i] * inv; }
    out->max_divb = r[16];
    out->enstrophy = r[20] * inv * inv; out->u2 = r[21] * inv * inv; out->current2 = r[24] * inv * inv;
    {
        const double den = out->u2 + out->emag;     // <|u|^2> + 1/2 <|B|^2>
        out->rayleigh_q = den > 0.0 ? (out->enstrophy + 0.5 * out->current2) / den : 0.0;
    }
    const bool bad = r[RED_NSUM] != 0.0 || r[17] != 0.0;
    if (bad) return fail(c, MHD_ENONFINITE, "non-finite value or rho <= 0 in the state");
    return MHD_OK;
}

}  // extern "C"

// ================================================================================================
// FFT-only entry points (BASELINE config 5).  Unpadded [batch][nz][ny][nx/2+1] layout, every mode
// kept.  R2C runs x (real -> out), then y and z in place in `out`; C2R runs z (in -> workspace),
// y in place, then x (workspace -> real), so the input is never written.
// ================================================================================================
struct mhd_fft_plan {
    int nx, ny, nz, batch, nxh;
    cudaStream_t st;
    int device;
    double2 *twx, *twy, *twz, *work;
    int plane;                 // x and y passes fused per plane through L2 (planefft_kernel.cu)
    int group, ring_slots, lag, pitch;
    double2* ring;
    unsigned* counters;
    char err[256];
};

namespace {
// plane pipeline geometry: groups of about 4 MB (>= 64 x-row items per group), the x pass 3 groups ahead of the y pass
#ifndef MHD_PF_LAG
#define MHD_PF_LAG 3
#endif
#ifndef MHD_PF_MINITEMS
#define MHD_PF_MINITEMS 64
#endif
struct PlaneGeom { int group, ring_slots, lag, pitch; };
PlaneGeom plane_geom(int n) {
    PlaneGeom g;
    const int tp = n / 8, teams = 512 / tp;
    const int per_plane = (n / 2 + teams - 1) / teams;
    g.group = (MHD_PF_MINITEMS + per_plane - 1) / per_plane;
    g.lag = MHD_PF_LAG;
    g.ring_slots = g.lag + 2;
    g.pitch = (n / 2 + 1 + 7) / 8 * 8;
    return g;
}
struct FftLayout { size_t twx, twy, twz, work, ring, counters, total; };
// with_ring: also the plane pipeline's ring and counters (only a plan that will use MHD_FFT_PLANE_PIPELINE pays for them);
// the layout without them is a prefix of the layout with them
FftLayout make_fft_layout(int nx, int ny, int nz, int batch, bool with_ring) {
    FftLayout L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
    L.twx = take(sizeof(double2) * nx); L.twy = take(sizeof(double2) * ny); L.twz = take(sizeof(double2) * nz);
    L.work = take(sizeof(double2) * (size_t)(nx / 2 + 1) * ny * nz * batch);
    L.ring = L.counters = o;
    if (with_ring && planefft_supported(nx, ny)) {
        const PlaneGeom g = plane_geom(nx);
        L.ring = take(sizeof(double2) * (size_t)g.ring_slots * g.group * ny * g.pitch);
        L.counters = take(planefft_counter_bytes((long long)batch * nz, g.group));
    }
    L.total = o;
    return L;
}
int pfail(mhd_fft_plan* p, const char* what, cudaError_t e) {
    snprintf(p->err, sizeof(p->err), "%s: %s", what, cudaGetErrorString(e));
    return MHD_ECUDA;
}
#define PCK(call)                                            \
    do {                                                     \
        cudaError_t e_ = (call);                             \
        if (e_ != cudaSuccess) return pfail(p, #call, e_);   \
    } while (0)
bool fft_dims_ok(int nx, int ny, int nz, int batch) {
    return fft_size_supported(nx) && fft_size_supported(ny) && (nz == 1 || fft_size_supported(nz)) && batch >= 1 && batch <= 4096;
}
}  // namespace

extern "C" {

size_t mhd_fft_workspace_bytes(int nx, int ny, int nz, int batch) {
    if (!fft_dims_ok(nx, ny, nz, batch)) return 0;
    return make_fft_layout(nx, ny, nz, batch, false).total;
}

size_t mhd_fft_plane_workspace_bytes(int nx, int ny, int nz, int batch) {
    if (!fft_dims_ok(nx, ny, nz, batch) || !planefft_supported(nx, ny)) return 0;
    return make_fft_layout(nx, ny, nz, batch, true).total;
}

int mhd_fft_plan_create(mhd_fft_plan** out, int nx, int ny, int nz, int batch, void* workspace, size_t bytes, void* stream) {
    if (!out) return MHD_EINVAL;
    *out = nullptr;
    if (!fft_dims_ok(nx, ny, nz, batch)) return MHD_EINVAL;
    FftLayout L = make_fft_layout(nx, ny, nz, batch, false);
    if (!workspace || bytes < L.total || ((size_t)workspace & 255u)) return MHD_EINVAL;
    const bool with_ring = planefft_supported(nx, ny) && bytes >= make_fft_layout(nx, ny, nz, batch, true).total;
    if (with_ring) L = make_fft_layout(nx, ny, nz, batch, true);
    mhd_fft_plan* p = new (std::nothrow) mhd_fft_plan();
    if (!p) return MHD_ENOMEM;
    p->err[0] = 0;
    p->device = owning_device(workspace);
    DeviceGuard guard(p->device);
    if (guard.failed) { delete p; return MHD_ECUDA; }
    if (!stream_on_device((cudaStream_t)stream, p->device)) { delete p; return MHD_EINVAL; }
    p->nx = nx; p->ny = ny; p->nz = nz; p->batch = batch; p->nxh = nx / 2 + 1; p->st = (cudaStream_t)stream;
    char* ws = (char*)workspace;
    p->twx = (double2*)(ws + L.twx); p->twy = (double2*)(ws + L.twy); p->twz = (double2*)(ws + L.twz); p->work = (double2*)(ws + L.work);
    p->plane = 0;              // default: three sweeps (faster on B200, see mhd_fft_plan_set_mode in mhd.h)
    p->ring = nullptr; p->counters = nullptr;
    if (with_ring) {
        const PlaneGeom g = plane_geom(nx);
        p->group = g.group; p->ring_slots = g.ring_slots; p->lag = g.lag; p->pitch = g.pitch;
        p->ring = (double2*)(ws + L.ring); p->counters = (unsigned*)(ws + L.counters);
    }
    std::vector<double2> t;
    const int n3[3] = {nx, ny, nz};
    double2* d3[3] = {p->twx, p->twy, p->twz};
    cudaError_t e = cudaSuccess;
    for (int a = 0; a < 3 && e == cudaSuccess; ++a) {
        host_twiddles(n3[a], t);
        e = cudaMemcpyAsync(d3[a], t.data(), sizeof(double2) * n3[a], cudaMemcpyHostToDevice, p->st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(p->st);
    }
    if (e != cudaSuccess) { delete p; return MHD_ECUDA; }
    *out = p;
    return MHD_OK;
}

void mhd_fft_plan_destroy(mhd_fft_plan* p) { delete p; }

int mhd_fft_plan_set_mode(mhd_fft_plan* p, int mode) {
    if (!p || (mode != MHD_FFT_THREE_SWEEP && mode != MHD_FFT_PLANE_PIPELINE)) return MHD_EINVAL;
    if (mode == MHD_FFT_PLANE_PIPELINE && !planefft_supported(p->nx, p->ny)) return MHD_EINVAL;
    if (mode == MHD_FFT_PLANE_PIPELINE && !p->ring) {
        snprintf(p->err, sizeof(p->err), "mhd_fft_plan_set_mode: the plan's workspace has no ring (create it with mhd_fft_plane_workspace_bytes)");
        return MHD_EINVAL;
    }
    p->plane = (mode == MHD_FFT_PLANE_PIPELINE) ? 1 : 0;
    return MHD_OK;
}

const char* mhd_fft_last_error(const mhd_fft_plan* p) { return p ? p->err : ""; }

int mhd_fft_r2c(mhd_fft_plan* p, const double* in, double* out) {
    if (!p || !in || !out) return MHD_EINVAL;
    DeviceGuard guard(p->device);
    if (guard.failed) { snprintf(p->err, sizeof(p->err), "%s", kGuardFailed); return MHD_ECUDA; }
    double2* o = (double2*)out;
    const long long plane = (long long)p->ny * p->nxh, vol = plane * p->nz;
    AxisArgs a;
    a.scale = 1.0;
    if (p->plane) {   // x and y in one persistent kernel, plane by plane through L2: the x-transformed rows never reach HBM
        PlaneFftArgs f;
        f.real = const_cast<double*>(in); f.spec_in = nullptr; f.spec_out = o; f.ring = p->ring; f.counters = p->counters;
        f.nplanes = (long long)p->batch * p->nz; f.group = p->group; f.ngroups = (f.nplanes + f.group - 1) / f.group;
        f.nxh = p->nxh; f.pitch = p->pitch; f.ring_slots = p->ring_slots; f.lag = p->lag; f.scale = 1.0;
        PCK(launch_planefft(p->nx, false, f, p->twx, p->st));
    } else {
        RowArgs r;
        r.spec = o; r.real = const_cast<double*>(in); r.spec_pitch = p->nxh; r.real_pitch = p->nx;
        r.nrows = (long long)p->batch * p->nz * p->ny; r.nkx = p->nxh; r.scale = 1.0;
        PCK(launch_fft_rows(p->nx, false, r, p->twx, p->st));
        a.in = o; a.out = o; a.nouter = (long long)p->batch * p->nz; a.in_outer = a.out_outer = plane;
        a.in_row = a.out_row = p->nxh; a.inner = p->nxh; a.nk_in = a.nk_out = p->ny;
        PCK(launch_fft_axis(p->ny, false, a, p->twy, p->st));
    }
    a.in = o; a.out = o;
    if (p->nz > 1) {
        a.nouter = p->batch; a.in_outer = a.out_outer = vol; a.in_row = a.out_row = plane;
        a.inner = (int)plane; a.nk_in = a.nk_out = p->nz;
        PCK(launch_fft_axis(p->nz, false, a, p->twz, p->st));
    }
    return MHD_OK;
}

int mhd_fft_c2r(mhd_fft_plan* p, const double* in, double* out) {
    if (!p || !in || !out) return MHD_EINVAL;
    DeviceGuard guard(p->device);
    if (guard.failed) { snprintf(p->err, sizeof(p->err), "%s", kGuardFailed); return MHD_ECUDA; }
    const double2* src = (const double2*)in;
    const long long plane = (long long)p->ny * p->nxh, vol = plane * p->nz;
    AxisArgs a;
    a.scale = 1.0;
    if (p->nz > 1) {
        a.in = src; a.out = p->work; a.nouter = p->batch; a.in_outer = a.out_outer = vol; a.in_row = a.out_row = plane;
        a.inner = (int)plane; a.nk_in = a.nk_out = p->nz;
        PCK(launch_fft_axis(p->nz, true, a, p->twz, p->st));
        src = p->work;
    }
    if (p->plane) {   // y and x in one persistent kernel, plane by plane through L2
        PlaneFftArgs f;
        f.real = out; f.spec_in = src; f.spec_out = nullptr; f.ring = p->ring; f.counters = p->counters;
        f.nplanes = (long long)p->batch * p->nz; f.group = p->group; f.ngroups = (f.nplanes + f.group - 1) / f.group;
        f.nxh = p->nxh; f.pitch = p->pitch; f.ring_slots = p->ring_slots; f.lag = p->lag;
        f.scale = 1.0 / ((double)p->nx * (double)p->ny * (double)p->nz);
        PCK(launch_planefft(p->nx, true, f, p->twx, p->st));
        return MHD_OK;
    }
    a.in = src; a.out = p->work; a.nouter = (long long)p->batch * p->nz; a.in_outer = a.out_outer = plane;
    a.in_row = a.out_row = p->nxh; a.inner = p->nxh; a.nk_in = a.nk_out = p->ny;
    PCK(launch_fft_axis(p->ny, true, a, p->twy, p->st));
    RowArgs r;
    r.spec = p->work; r.real = out; r.spec_pitch = p->nxh; r.real_pitch = p->nx;
    r.nrows = (long long)p->batch * p->nz * p->ny; r.nkx = p->nxh;
    r.scale = 1.0 / ((double)p->nx * (double)p->ny * (double)p->nz);
    PCK(launch_fft_rows(p->nx, true, r, p->twx, p->st));
    return MHD_OK;
}

}  // extern "C"
