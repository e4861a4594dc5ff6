/* mhd.h — C ABI of the B200 (sm_100a) pseudo-spectral isothermal MHD step.
 *
 * What it computes (arxiv 2402.05478, PAPER.md):
 *   eq. (1) PAPER.md:39   d rho/dt + div(rho u) = 0
 *   eq. (2) PAPER.md:41   d(rho u)/dt + div[rho u u + (P + B^2/2) I - B B] = (1/Re) lap u   (f = 0)
 *   eq. (3) PAPER.md:45   P = Cs^2 rho
 *   eq. (4) PAPER.md:47   dB/dt + div(u B - B u) = (1/Rm) lap B      ( = curl(u x B) + eta lap B )
 * discretised as PAPER.md:78 describes: Fourier pseudo-spectral on a triply periodic box [0,2pi)^3,
 * derivatives by i*k in Fourier space, products in real space, "standard 2/3 de-aliasing rule",
 * Adams-Bashforth time stepping (AB2 with a forward-Euler first step) or Runge-Kutta 4
 * (Table II), double precision.  Evolved variables are rho, m = rho u
 * and B as spectral coefficients; the caller sees rho, u, B on the grid.
 *
 * Everything runs on ONE GPU in hand-written CUDA kernels (own FFT; no cuFFT, no CPU fallback).
 * The library never allocates or frees device memory: the caller passes a workspace (e.g. a torch
 * tensor) and a CUDA stream; all work is enqueued on that stream.
 *
 * Layouts.  Real fields: nx*ny*nz doubles, index ((z*ny + y)*nx + x), x fastest, x_j = 2*pi*j/nx.
 * Half-spectra (FFT entry points only): [batch][nz][ny][nx/2+1] complex, re/im interleaved,
 * kx = 0..nx/2 fastest, ky / kz in FFT order.  Forward transform f^(k) = sum_x f(x) exp(-i k.x),
 * unnormalised; the inverse includes 1/(nx*ny*nz).
 *
 * Sizes: nx, ny in {8,12,16,24,32,48,64,96,128,192,256,384,512,768,1024}; nz from the same set or
 * nz == 1 (2-D run: the z transform is the identity and kz = 0).
 *
 * Pointers named *_dev are DEVICE pointers, *_host are HOST pointers (pinned memory makes the
 * copies asynchronous, pageable memory works too).  Every call returns MHD_OK or a negative code;
 * nothing throws, aborts or prints.  Invalid arguments are rejected before any launch.  A context
 * is not thread-safe; distinct contexts are independent, also on different devices of one process: every
 * call makes the device that owns the context's workspace current for its own duration and restores the caller's.
 * Results are bit-reproducible run to run (no floating-point atomics).
 */
#ifndef MHD_H
#define MHD_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mhd_ctx mhd_ctx;            /* opaque; host memory owned by the library, freed by mhd_destroy */
typedef struct mhd_fft_plan mhd_fft_plan;  /* opaque */

enum { MHD_OK = 0, MHD_EINVAL = -1, MHD_ENOMEM = -2, MHD_ECUDA = -3, MHD_ESTATE = -4, MHD_ENONFINITE = -5 };
enum { MHD_AB2 = 0, MHD_RK4 = 1 };
enum {
    MHD_FLAG_HYDRO = 1u,      /* B == 0 held exactly: induction and Lorentz terms skipped */
    MHD_FLAG_NO_DEALIAS = 2u, /* keep every mode (tests only) */
    MHD_FLAG_FORCING = 4u,    /* reserve workspace for the steady body force f of eq. (2) (mhd_set_forcing) */
    /* Execution-plan switches.  They never change what is computed (results agree to roundoff with the default plan and are
     * covered by the same parity tests); they exist so that every kernel of the library can be reached, tested and timed
     * through this ABI.  Nothing in the library reads the environment. */
    MHD_FLAG_UNFUSED_X = 8u,      /* x C2R, real-space products and x R2C as three kernels through real arrays, instead of the
                                     fused x pass (the plan that nx = 3*2^a always uses: the fused pass needs 8 points per thread) */
    MHD_FLAG_NO_GRAPH = 16u       /* mhd_step always enqueues its kernels one by one (no CUDA-graph replay) */
};

/* mean values are volume averages <.> = (1/N) sum over the grid */
typedef struct {
    long long step;    /* steps taken since mhd_set_fields */
    double time;       /* step * dt */
    double ekin;       /* 1/2 <rho |u|^2> */
    double emag;       /* 1/2 <|B|^2>               (eq. 2) */
    double eiso;       /* Cs^2 <rho ln rho>: ekin+emag+eiso is the ideal invariant of the isothermal system */
    double mass;       /* <rho> */
    double mom[3];     /* <rho u> */
    double bmean[3];   /* <B> */
    double max_divb;   /* max_x |IFFT(i k . B^)| */
    /* the paper's diagnostics, as sums over the spectra of u = m/rho (every mode, not only the retained ones) and B: */
    double enstrophy;  /* <|curl u|^2> = sum_k |k x u^|^2 / N^2: mean-square vorticity Omega(t) */
    double current2;   /* <|curl B|^2> = sum_k |k x B^|^2 / N^2 */
    double u2;         /* <|u|^2> */
    double rayleigh_q; /* (enstrophy + current2/2) / (u2 + <|B|^2>/2): Rayleigh quotient Q(t), eq. (14) */
} mhd_diag;

/* Bytes of device workspace mhd_create needs for this configuration (0 if the size is unsupported). */
size_t mhd_workspace_bytes(int nx, int ny, int nz, int integrator, unsigned flags);

/* Create a context.  nu = 1/Re, eta = 1/Rm, cs = sound speed (all >= 0), dt > 0.
 * workspace_dev: caller-owned device memory, 256-byte aligned, >= mhd_workspace_bytes(...), must stay
 * alive and untouched until mhd_destroy.  cuda_stream: a cudaStream_t; NULL = the legacy default
 * stream, on which mhd_step cannot use CUDA graphs (small grids then pay per-launch latency).
 * Errors: MHD_EINVAL (bad size/parameter/NULL/workspace too small, or cuda_stream was created on another GPU than the one
 * that owns the workspace), MHD_ENOMEM (host), MHD_ECUDA.  Any later call returns MHD_ECUDA, without launching anything, if
 * the GPU that owns the workspace cannot be made current. */
int mhd_create(mhd_ctx** out, int nx, int ny, int nz, double nu, double eta, double cs, double dt,
               int integrator, unsigned flags, void* workspace_dev, size_t workspace_bytes, void* cuda_stream);
void mhd_destroy(mhd_ctx* ctx);

/* Box lengths (the KH test uses Lx = 1, Ly = 2; every other test the 2*pi box): wavenumbers become
 * k_i = 2*pi*n_i/L_i.  Default 2*pi per axis (k = n exactly).  The 2/3 mask stays a test on the integers n_i; lz is
 * ignored when nz == 1.  May be called at any time; takes effect from the next mhd_step / mhd_diagnostics.
 * MHD_EINVAL unless every length is finite and > 0. */
int mhd_set_box(mhd_ctx* ctx, double lx, double ly, double lz);

/* Steady body force f(x) of eq. (2) ("+ f"; App. B eqs B2-B3), nx*ny*nz doubles per
 * component on the grid (DEVICE pointers; the _host variant takes HOST pointers).  Its 2/3-masked transform is kept
 * in the workspace and added to the momentum right-hand side of every later step.  NULL, NULL, NULL switches it off.
 * Needs MHD_FLAG_FORCING at mhd_create (MHD_ESTATE otherwise).  Asynchronous; inputs are read, never written. */
int mhd_set_forcing(mhd_ctx* ctx, const double* fx_dev, const double* fy_dev, const double* fz_dev);
int mhd_set_forcing_host(mhd_ctx* ctx, const double* fx_host, const double* fy_host, const double* fz_host);

/* Set the state from grid fields: m = rho*u, forward transform, 2/3 mask.
 * Resets step count, time and integrator history.  b* may be NULL with MHD_FLAG_HYDRO.
 * Asynchronous on the context's stream; inputs are read, never written. */
int mhd_set_fields(mhd_ctx* ctx, const double* rho_dev, const double* ux_dev, const double* uy_dev,
                   const double* uz_dev, const double* bx_dev, const double* by_dev, const double* bz_dev);
/* Same from HOST arrays: copies host->device into the workspace on the stream, then as above. */
int mhd_set_fields_host(mhd_ctx* ctx, const double* rho_host, const double* ux_host, const double* uy_host,
                        const double* uz_host, const double* bx_host, const double* by_host, const double* bz_host);

/* Advance nsteps >= 0 time steps (one RHS evaluation per AB2 step, four per RK4 step).
 * Asynchronous: enqueues and returns.  MHD_ESTATE before the first mhd_set_fields. */
int mhd_step(mhd_ctx* ctx, int nsteps);

/* Current rho, u = m/rho, B on the grid, into caller-owned DEVICE (or HOST) arrays; b* may be NULL.
 * The device variant is asynchronous; the host variant returns after the copies have completed. */
int mhd_get_fields(mhd_ctx* ctx, double* rho_dev, double* ux_dev, double* uy_dev, double* uz_dev,
                   double* bx_dev, double* by_dev, double* bz_dev);
int mhd_get_fields_host(mhd_ctx* ctx, double* rho_host, double* ux_host, double* uy_host, double* uz_host,
                        double* bx_host, double* by_host, double* bz_host);

/* Diagnostics of the current state into HOST memory; synchronises the stream.
 * Spectra (optional, nshell may be 0): shell s = round(|k|), s = 0..nshell-1,
 *   ekin_spec[s] = sum_{k in s} 1/2 |u^(k)|^2 / N^2   with u = m/rho (sums to 1/2 <|u|^2>),
 *   emag_spec[s] = sum_{k in s} 1/2 |B^(k)|^2 / N^2   (sums to emag).
 * Spectra are defined on the 2*pi box only (MHD_EINVAL with nshell > 0 after mhd_set_box to another length).
 * Returns MHD_ENONFINITE (values still filled) if a NaN/Inf or rho <= 0 was seen, MHD_ECUDA on a
 * sticky CUDA error. */
int mhd_diagnostics(mhd_ctx* ctx, mhd_diag* out_host, double* ekin_spec_host, double* emag_spec_host, int nshell);

/* Exact resume (the paper restarts from ASCII dumps; restarting AB2 from grid fields alone would
 * re-bootstrap with an Euler step).  mhd_get_state copies the spectral state, the integrator history and a small header
 * (grid, flags, integrator, step count) into state_dev, a caller-owned DEVICE buffer of mhd_state_bytes(ctx) bytes;
 * mhd_set_state restores them into a context created with the same nx, ny, nz, integrator and flags (MHD_EINVAL
 * otherwise; it synchronises to read the header).  A run continued after mhd_set_state is bit-identical to the
 * uninterrupted run.  The blob's layout is internal to this library version.  Box, forcing, nu, eta, cs, dt are NOT
 * part of the state: set them on the new context as before. */
size_t mhd_state_bytes(const mhd_ctx* ctx);
int mhd_get_state(mhd_ctx* ctx, void* state_dev, size_t bytes);
int mhd_set_state(mhd_ctx* ctx, const void* state_dev, size_t bytes);

const char* mhd_strerror(int code);
const char* mhd_last_error(const mhd_ctx* ctx);   /* detail of the last failure on this context ("" if none) */

/* ---- FFT-only entry points (BASELINE config 5: batched 3-D R2C / C2R throughput) ---------------- */
size_t mhd_fft_workspace_bytes(int nx, int ny, int nz, int batch);
int  mhd_fft_plan_create(mhd_fft_plan** out, int nx, int ny, int nz, int batch,
                         void* workspace_dev, size_t workspace_bytes, void* cuda_stream);
/* in_real_dev: [batch][nz][ny][nx] doubles; out_complex_dev: [batch][nz][ny][nx/2+1] complex; unnormalised */
int  mhd_fft_r2c(mhd_fft_plan* plan, const double* in_real_dev, double* out_complex_dev);
/* inverse, includes 1/(nx*ny*nz); Im of self-conjugate x modes (kx = 0, nx/2 of a row) is ignored */
int  mhd_fft_c2r(mhd_fft_plan* plan, const double* in_complex_dev, double* out_real_dev);
void mhd_fft_plan_destroy(mhd_fft_plan* plan);
/* How the x and y passes run.  MHD_FFT_THREE_SWEEP (default): one kernel per axis, every pass streams the batch through HBM
 * (6 F of traffic per transform).  MHD_FFT_PLANE_PIPELINE (square planes nx == ny in {64,128,256,512} only, MHD_EINVAL
 * otherwise): x and y passes in one persistent kernel, plane groups handed over through an L2-resident ring (4 F of traffic:
 * the "2-sweep" transform of SURVEY.md §8(f) #4).  Same results to roundoff.  Measured on B200 at 512^3: DRAM traffic of the x+y
 * part falls from 30 GB to 15 GB, but the kernel is bound by the SM's load-store pipe, not by HBM, and runs slower than
 * the two separate passes (profiles/r02_planefft.md): hence not the default. */
enum { MHD_FFT_THREE_SWEEP = 0, MHD_FFT_PLANE_PIPELINE = 1 };
int mhd_fft_plan_set_mode(mhd_fft_plan* plan, int mode);
/* The plane pipeline needs a ring of plane groups and its counters behind the plan's ordinary workspace (about 20 MB).  Only a
 * plan that will use it pays: mhd_fft_workspace_bytes does not include them; a plan created on at least
 * mhd_fft_plane_workspace_bytes(...) bytes (0 for shapes the mode does not take) may switch to MHD_FFT_PLANE_PIPELINE, any
 * smaller plan gets MHD_EINVAL from mhd_fft_plan_set_mode. */
size_t mhd_fft_plane_workspace_bytes(int nx, int ny, int nz, int batch);
const char* mhd_fft_last_error(const mhd_fft_plan* plan);   /* detail of the last MHD_ECUDA on this plan ("" if none) */

/* ---- The inverse transform without a workspace -------------------------------------------------------------------
 * mhd_fft_c2r computes out = C2R(in) through a plan, and a plan needs device memory from the caller (twiddle tables and one
 * half-spectrum-sized intermediate, since `in` is never written).  A caller that owns its input and output and cannot get
 * any more device memory -- a callback inside a framework whose allocator already holds the whole GPU, a job whose fixed
 * memory budget is fully handed out, a loop that may not call cudaMalloc because cudaMalloc synchronises the device --
 * calls this instead.  Same transform, same layouts, same kernels and twiddle values as mhd_fft_c2r (plan of nx, ny, nz,
 * batch in the default three-sweep mode): in_complex_dev [batch][nz][ny][nx/2+1] complex, read only; out_real_dev
 * [batch][nz][ny][nx] doubles; includes 1/(nx*ny*nz).  Both are DEVICE pointers on the same GPU; the call runs on the GPU
 * that owns out_real_dev, enqueued on cuda_stream (NULL = legacy default stream), and is asynchronous after the first call.
 *
 * The scratch is an array compiled into the library: MHD_STATIC_SCRATCH_BYTES for the intermediate plus 56 KiB of twiddle
 * tables.  Every GPU that loads the library holds it until the process exits, used or not, which is why it is small.
 * The call allocates and frees nothing on the device.  A transform whose intermediate, 16*(nx/2+1)*ny*nz*batch bytes,
 * exceeds MHD_STATIC_SCRATCH_BYTES (64^3 x 3, 96^3, 512^2 x 3 fit; 128^3 does not) is refused with MHD_EINVAL before
 * anything is launched, and err_host says how much was asked for and how much there is.
 *
 * First call on each GPU: looks up the array's device address, uploads the twiddle tables and synchronises cuda_stream
 * (a few hundred microseconds).  Make that call before you begin any stream capture on that GPU; a 8x8x8 transform will do.
 * One array per GPU, shared by every call: two calls that can run at the same time on one GPU (different streams, or
 * different host threads without a common stream) overwrite each other's intermediate -- keep them on one stream or order
 * them yourself.  The array keeps the previous call's contents; nothing in it has to start at zero, because every element a
 * call reads it has written earlier in the same call, so nothing is cleared.
 *
 * err_host: optional HOST buffer of err_bytes for a one-line description of a failure ("" on success); may be NULL.
 * Returns MHD_OK, MHD_EINVAL (unsupported length, NULL buffer, too large) or MHD_ECUDA. */
#define MHD_STATIC_SCRATCH_BYTES (8u << 20)
int mhd_fft_c2r_static(int nx, int ny, int nz, int batch, const double* in_complex_dev, double* out_real_dev,
                       void* cuda_stream, char* err_host, size_t err_bytes);

/* ==== Instrumentation (not part of the solver's contract; used by bench.py and the tests) ====================== */

/* number of kernel launches this library has enqueued since load (bench.py's gpu_launches) */
long long mhd_launch_count(void);

/* Per-kernel timing for the roofline report.  After mhd_profile_begin, mhd_step runs its kernels
 * eagerly with a CUDA-event pair around every launch (on the context's stream); mhd_profile_end
 * synchronises, fills counts[i] (launches) and ms[i] (summed device time) for the
 * mhd_profile_kernel_count() kernel classes named by mhd_profile_kernel_name(i) -- in hot-path
 * order: z inverse, y inverse, x C2R, products, x R2C, fused x pass, y forward, z forward, stage (its two launches, (rho, m)
 * and B, counted as one) -- and switches
 * profiling off.  Both arrays are HOST memory of that length. */
int mhd_profile_kernel_count(void);
const char* mhd_profile_kernel_name(int i);
int mhd_profile_begin(mhd_ctx* ctx);
int mhd_profile_end(mhd_ctx* ctx, int* counts_host, double* ms_host);

/* Measured ceilings of the on-chip resources that bound the fused x pass ("FP64 peak is nominal --
 * builder to measure"): the FP64 FMA pipe (TFLOP/s, a DFMA = 2 flop, independent register-only chains) and the
 * shared-memory data path (GB/s moved between shared memory and registers by conflict-free 16-byte accesses).
 * scratch_dev: DEVICE memory of scratch_bytes >= 4 MiB on the current device; synchronises; results in HOST doubles. */
int mhd_measure_peaks(void* scratch_dev, size_t scratch_bytes, void* cuda_stream, double* fp64_tflops_host, double* smem_gbs_host);

/* What the fused x pass's own shared-memory exchange pattern reaches with everything else stripped away: 4 teams of 64 threads
 * per SM, per iteration dfma_per_exchange (0, 64, 128, 192 or 256) independent DFMAs per thread, then 16 STS.128 and 16 LDS.128
 * (the padded index sets of the Stockham passes) with team barriers placed by barrier_mode: 0 = write, barrier, read, barrier;
 * 1 = barrier, write, barrier, read (the shipped x passes); 2 = two buffers used alternately, one barrier per exchange;
 * 3 = no shared memory at all: the same 16 complex values per thread exchanged by an 8 x 8 register transpose among the 8 lanes
 * of a warp octet (three __shfl_xor_sync rounds) -- the upper bound of a warp-shuffle exchange, reported in the same unit
 * (512 bytes per thread and exchange) so that it can be read against the shared-memory modes.
 * Result: GB/s moved through shared memory.  The fused pass at N = 512 has ~190 FP64 instructions per thread between
 * exchanges; its achievable ceiling is this number, not the free-running shared-memory peak of mhd_measure_peaks.
 * scratch_dev as above; synchronises; MHD_EINVAL for other counts or modes. */
int mhd_measure_exchange(void* scratch_dev, size_t scratch_bytes, void* cuda_stream, int dfma_per_exchange, int barrier_mode,
                         double* smem_gbs_host);

#ifdef __cplusplus
}
#endif
#endif
