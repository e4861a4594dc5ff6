// fft_c2r_static.cu — mhd_fft_c2r_static (include/mhd.h): the batched 3-D complex-to-real transform of mhd_fft_c2r for a
// caller that has no way of getting device memory for a plan workspace.
//
// Who that is.  mhd_fft_c2r needs a plan, and a plan needs a caller-supplied workspace (twiddle tables plus one
// half-spectrum-sized intermediate, because the input must not be written).  Some callers own their input and output
// buffers and nothing else: a callback running inside another framework whose allocator holds the whole GPU (a raw
// cudaMalloc there fails or fragments the pool), a process confined to a fixed memory budget that has been handed out in
// full, a latency-critical loop that may not call cudaMalloc because it synchronises the device.  For them the scratch lives
// in the library image itself: the file-scope array below.  It is reserved on every GPU that loads this library, from the
// moment the module is loaded until the process exits, whether or not this entry point is ever called; that is why it is
// kept small (MHD_STATIC_SCRATCH_BYTES for the intermediate + 56 KiB of twiddle tables).
//
// Nothing here calls cudaMalloc, cudaFree or a library routine that allocates device memory.  The kernels are the ones
// mhd_fft_c2r launches (launch_fft_axis / launch_fft_rows), with the same twiddle values, so results are the same.
#include "../../include/mhd.h"
#include "mhd_internal.h"

#include <math.h>
#include <stdio.h>

#include <mutex>

using namespace mhd;

namespace {

// twiddle tables for every supported axis length, each starting on a 256-byte boundary (16 complex)
constexpr int kNumSizes = 15;
constexpr int kSizes[kNumSizes] = {8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024};
constexpr size_t table_slot(int n) { return ((size_t)n + 15) / 16 * 16; }
constexpr size_t tables_total() {
    size_t t = 0;
    for (int i = 0; i < kNumSizes; ++i) t += table_slot(kSizes[i]);
    return t;
}
constexpr size_t kTableComplex = tables_total();                              // 3584 complex = 56 KiB
constexpr size_t kWorkComplex = (size_t)MHD_STATIC_SCRATCH_BYTES / sizeof(double2);

// The scratch.  In HOST code this name is only a handle for the runtime (cudaGetSymbolAddress below turns it into the device
// address, per device); it must never be passed to a kernel as a pointer.  Layout: [twiddle tables][intermediate].
static __device__ __align__(256) double2 g_static_scratch[kTableComplex + kWorkComplex];

struct DeviceScratch {
    bool ready;
    double2* base;      // device address of g_static_scratch on this device
};
DeviceScratch g_dev[kMaxDevices];
std::mutex g_setup_mutex;
double2 g_host_tables[kTableComplex];   // host staging for the one upload per device (guarded by g_setup_mutex)

size_t table_offset(int n) {
    size_t o = 0;
    for (int i = 0; i < kNumSizes; ++i) {
        if (kSizes[i] == n) return o;
        o += table_slot(kSizes[i]);
    }
    return (size_t)-1;
}

// exp(-2 pi i j / n) in long double, rounded once: the values mhd_fft_plan_create puts into a plan workspace
void fill_table(int n, double2* t) {
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int j = 0; j < n; ++j) {
        const long double a = two_pi * (long double)j / (long double)n;
        t[j] = make_double2((double)cosl(a), -(double)sinl(a));
    }
}

// Once per device, with that device current: find where the array lives on this GPU and fill the twiddle tables.
cudaError_t setup_device(int dev, cudaStream_t st, double2** base) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (g_dev[dev].ready) { *base = g_dev[dev].base; return cudaSuccess; }
    double2* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    for (size_t i = 0; i < kTableComplex; ++i) g_host_tables[i] = make_double2(0.0, 0.0);
    for (int i = 0; i < kNumSizes; ++i) fill_table(kSizes[i], g_host_tables + table_offset(kSizes[i]));
    e = cudaMemcpyAsync(p, g_host_tables, sizeof(double2) * kTableComplex, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);      // the staging array is reused by the next device's set-up
    if (e != cudaSuccess) return e;
    g_dev[dev].base = p;
    g_dev[dev].ready = true;
    *base = p;
    return cudaSuccess;
}

// runs the call on the GPU that owns the output buffer, whatever device the calling thread has current
struct CurrentDevice {
    int prev = -1;
    bool switched = false;
    explicit CurrentDevice(const void* p) {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return; }
        if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != at.device) switched = (cudaSetDevice(at.device) == cudaSuccess);
    }
    ~CurrentDevice() {
        if (switched) cudaSetDevice(prev);
    }
};

int report(char* err, size_t err_bytes, int code, const char* msg) {
    if (err && err_bytes > 0) snprintf(err, err_bytes, "%s", msg);
    return code;
}

}  // namespace

extern "C" int mhd_fft_c2r_static(int nx, int ny, int nz, int batch, const double* in_complex_dev, double* out_real_dev,
                                  void* cuda_stream, char* err_host, size_t err_bytes) {
    char msg[256];
    if (err_host && err_bytes > 0) err_host[0] = 0;
    if (!fft_size_supported(nx) || !fft_size_supported(ny) || (nz != 1 && !fft_size_supported(nz)) || batch < 1 || batch > 4096) {
        snprintf(msg, sizeof(msg), "mhd_fft_c2r_static: unsupported size %d x %d x %d, batch %d", nx, ny, nz, batch);
        return report(err_host, err_bytes, MHD_EINVAL, msg);
    }
    if (!in_complex_dev || !out_real_dev) return report(err_host, err_bytes, MHD_EINVAL, "mhd_fft_c2r_static: NULL input or output");
    const int nxh = nx / 2 + 1;
    const unsigned long long need = 16ull * (unsigned long long)nxh * ny * nz * batch;      // one half-spectrum intermediate
    if (need > (unsigned long long)MHD_STATIC_SCRATCH_BYTES) {
        snprintf(msg, sizeof(msg),
                 "mhd_fft_c2r_static: %d x %d x %d, batch %d needs %llu bytes of scratch; the built-in array holds %llu "
                 "(use a plan with mhd_fft_c2r for larger transforms)",
                 nx, ny, nz, batch, need, (unsigned long long)MHD_STATIC_SCRATCH_BYTES);
        return report(err_host, err_bytes, MHD_EINVAL, msg);
    }
    CurrentDevice on(out_real_dev);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int dev = device_slot();
    if (dev < 0) return report(err_host, err_bytes, MHD_ECUDA, "mhd_fft_c2r_static: no current CUDA device");
    double2* base = nullptr;
    cudaError_t e = setup_device(dev, st, &base);
    const char* where = "set-up (cudaGetSymbolAddress / twiddle upload)";
    if (e == cudaSuccess) {
        const double2* twx = base + table_offset(nx);
        const double2* twy = base + table_offset(ny);
        const double2* twz = base + table_offset(nz == 1 ? nx : nz);      // unused when nz == 1
        double2* work = base + kTableComplex;
        const double2* src = (const double2*)in_complex_dev;
        const long long plane = (long long)ny * nxh, vol = plane * nz;
        AxisArgs a;
        a.scale = 1.0;
        if (nz > 1) {       // z: input -> intermediate
            a.in = src; a.out = work; a.nouter = batch; a.in_outer = a.out_outer = vol; a.in_row = a.out_row = plane;
            a.inner = (int)plane; a.nk_in = a.nk_out = nz;
            where = "z pass";
            e = launch_fft_axis(nz, true, a, twz, st);
            src = work;
        }
        if (e == cudaSuccess) {   // y: in place in the intermediate (from the input when there is no z pass)
            a.in = src; a.out = work; a.nouter = (long long)batch * nz; a.in_outer = a.out_outer = plane;
            a.in_row = a.out_row = nxh; a.inner = nxh; a.nk_in = a.nk_out = ny;
            where = "y pass";
            e = launch_fft_axis(ny, true, a, twy, st);
        }
        if (e == cudaSuccess) {   // x: half-spectrum rows -> real rows of the output
            RowArgs r;
            r.spec = work; r.real = out_real_dev; r.spec_pitch = nxh; r.real_pitch = nx;
            r.nrows = (long long)batch * nz * ny; r.nkx = nxh;
            r.scale = 1.0 / ((double)nx * (double)ny * (double)nz);
            where = "x pass";
            e = launch_fft_rows(nx, true, r, twx, st);
        }
    }
    if (e != cudaSuccess) {
        snprintf(msg, sizeof(msg), "mhd_fft_c2r_static: %s: %s", where, cudaGetErrorString(e));
        return report(err_host, err_bytes, MHD_ECUDA, msg);
    }
    return MHD_OK;
}
