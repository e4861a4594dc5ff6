// mhd_internal.h — declarations shared by the CUDA translation units of libmhd_b200 (not public).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace mhd {

// ---- FFT launch arguments ------------------------------------------------------------------
struct AxisArgs {                 // transform along a strided axis of [outer][rows][inner] complex
    const double2* in;
    double2* out;
    long long nouter;             // number of outer slabs
    long long in_outer, out_outer;  // slab strides (complex elements)
    long long in_row, out_row;      // strides between consecutive rows of the axis
    int inner;                    // contiguous columns per row
    int nk_in, nk_out;            // rows stored: N (all) or 2*kmax+1 (compact, 2/3 rule)
    double scale;                 // applied on store
};
struct RowArgs {                  // x axis: half-spectrum rows <-> real rows
    double2* spec;
    double* real;
    long long spec_pitch;         // complex elements between rows
    long long real_pitch;         // doubles between rows
    long long nrows;              // even
    int nkx;                      // complex stored per row: nx/2+1 or kmax+1
    double scale;
};

bool fft_size_supported(int n);
cudaError_t launch_fft_axis(int n, bool inverse, const AxisArgs& a, const double2* tw, cudaStream_t st);
cudaError_t launch_fft_rows(int n, bool inverse, const RowArgs& a, const double2* tw, cudaStream_t st);

// ---- x and y passes of a batched 3-D real FFT in one persistent kernel, plane by plane through L2 (planefft_kernel.cu) ----
struct PlaneFftArgs {
    double* real;             // [nplanes][n][n] doubles: input (forward) or output (inverse)
    const double2* spec_in;   // inverse: [nplanes][n][nxh] half-spectrum planes (y not yet transformed)
    double2* spec_out;        // forward: [nplanes][n][nxh] half-spectrum planes (x and y transformed)
    double2* ring;            // ring_slots * group planes of n * pitch complex (the L2-resident intermediate)
    unsigned* counters;       // planefft_counter_bytes(...) bytes, 8-byte aligned; zeroed by the launcher
    long long nplanes, ngroups;
    int nxh, pitch;           // n/2+1 and the ring's row pitch (multiple of 8)
    int group, ring_slots, lag;
    double scale;             // applied by the inverse x pass
};
bool planefft_supported(int nx, int ny);
size_t planefft_counter_bytes(long long nplanes, int group);
cudaError_t launch_planefft(int n, bool inverse, const PlaneFftArgs& a, const double2* tw, cudaStream_t st);

// ---- fused x pass (xfused_kernel.cu): C2R-x -> products -> R2C-x, in place on [field][row][px] ----
struct XFusedArgs {
    double2* w2;              // inputs: fields 0..6 (0..3 hydro); outputs: product fields 0..11 (0..8 hydro)
    long long field_stride;   // complex elements per field
    long long nrows;          // nz*ny
    int px, nkx;              // row pitch and stored modes per row
    double scale;             // 1/(nx*ny*nz), applied to the inverse transforms
};
bool xfused_supported(int n);
// stand-alone x pass (row pairs) on the fused kernel's team machinery; n must satisfy xfused_supported(n)
cudaError_t launch_xrows(int n, bool inverse, const RowArgs& a, const double2* tw, cudaStream_t st);
cudaError_t launch_xfused(int n, const XFusedArgs& a, int hydro, const double2* tw, cudaStream_t st);

// ---- pointwise / spectral kernels (mhd_kernels.cu) ------------------------------------------
// real-space field order in a block of consecutive arrays (stride = points per field)
enum { F_RHO = 0, F_MX, F_MY, F_MZ, F_BX, F_BY, F_BZ, NFIELD = 7 };
// product order: u first so that the hydro run uses the first 9 only
enum { P_UX = 0, P_UY, P_UZ, P_TXX, P_TYY, P_TZZ, P_TXY, P_TXZ, P_TYZ, P_EX, P_EY, P_EZ, NPROD = 12 };

struct SpecGeom {                 // compact spectral array [nkz][nky][px]
    int nx, ny, nz;               // grid
    int nkx, nky, nkz;            // stored modes per axis
    int px;                       // row pitch in complex elements (multiple of 8)
    long long field;              // complex elements per field = nkz*nky*px
};

// stage update modes
enum { STAGE_AB2_EULER = 0, STAGE_AB2 = 1, STAGE_RK4_1 = 2, STAGE_RK4_2 = 3, STAGE_RK4_3 = 4, STAGE_RK4_4 = 5 };

struct StageArgs {
    SpecGeom g;
    double2* S;                   // 7 fields: state read by the RHS (and written, see mode)
    const double2* G;             // 12 (9 hydro) flux fields
    double2* H;                   // AB2: previous RHS (7 fields).  RK4: S0 (state at step start)
    double2* Acc;                 // RK4: accumulator (7 fields)
    const double2* F;             // masked transform of the body force (3 fields) or nullptr
    double nu, eta, cs2, dt;
    double kfx, kfy, kfz;         // 2*pi/L per axis: physical wavenumber = factor * integer index
    int mode;
    int hydro;
};

cudaError_t launch_products(const double* f, double* g, long long npts, int hydro, cudaStream_t st);
cudaError_t launch_stage(const StageArgs& a, cudaStream_t st);
cudaError_t launch_momentum(const double* rho, const double* ux, const double* uy, const double* uz, double* m,
                            long long npts, cudaStream_t st);            // m_i = rho*u_i into 3 consecutive fields
cudaError_t launch_velocity(const double* f, double* ux, double* uy, double* uz, long long npts, cudaStream_t st);
cudaError_t launch_velocity3(const double* f, double* u3, long long npts, cudaStream_t st);  // u = m/rho, 3 consecutive
cudaError_t launch_divb_spec(const SpecGeom& g, const double2* B, double2* out, double kfx, double kfy, double kfz, cudaStream_t st);  // i k.B^
// results[0] = sum_k w |k x V^|^2, results[1] = sum_k w |V^|^2 over the full spectrum (w = 1 on self-conjugate x planes, else 2)
cudaError_t launch_reduce_curl(const SpecGeom& g, const double2* V3, double kfx, double kfy, double kfz, double* partial, double* results, cudaStream_t st);
cudaError_t launch_zero(void* p, size_t bytes, cudaStream_t st);

// reductions: results[0..9] = sums of (ekin, emag, rho ln rho, rho, mx, my, mz, bx, by, bz) terms, results[10] = bad flag
enum { RED_NSUM = 10, RED_BLOCKS = 1184 };   // 8 x 148 blocks, fixed => deterministic
cudaError_t launch_reduce_fields(const double* f, long long npts, int hydro, double* partial, double* results, cudaStream_t st);
cudaError_t launch_reduce_maxabs(const double* a, long long npts, double* partial, double* result, cudaStream_t st);
// shell spectra (deterministic): rows -> per-row run sums -> per-shell gather
cudaError_t launch_spectrum(const SpecGeom& g, const double2* V3, double* rowbins, double* spec, int nshell, cudaStream_t st);

void count_launch();
long long launch_count();
void add_launches(long long n);

// ---- instrumentation: measured FP64-FMA and shared-memory ceilings (peaks_kernel.cu) ----
cudaError_t measure_peaks(double* scratch, size_t scratch_doubles, cudaStream_t st, double* fp64_tflops, double* smem_gbs);
// shared-memory GB/s of the fused x pass's exchange pattern (team barriers, bursts of 16 + 16 accesses) with dfma_per_exchange
// (0, 64, ..., 256) DFMAs per thread in between
// mode: 0 write-barrier-read-barrier, 1 barrier-write-barrier-read (shipped), 2 double-buffered, one barrier per exchange
cudaError_t measure_exchange(double* scratch, size_t scratch_doubles, cudaStream_t st, int dfma_per_exchange, int mode, double* smem_gbs);

// ---- per-device one-time kernel setup ---------------------------------------------------------------
// cudaFuncSetAttribute (opt-in dynamic shared memory) and the SM count belong to a DEVICE, not to the process: every
// launcher keeps one DeviceOnce per kernel family and asks it for the current device's slot.
constexpr int kMaxDevices = 64;
struct DeviceOnce {
    bool done[kMaxDevices];
    int sms[kMaxDevices];
};
// index of the calling thread's current device in a DeviceOnce (cudaGetDevice), or -1 on error / out of range
int device_slot();
// SM count of device slot `dev` (cached per device)
cudaError_t device_sm_count(int dev, int* sms);

}  // namespace mhd
