// fft_kernels.cu — batched pencil-FFT kernels for sm_100a (fp64), built on fft_core.cuh.
//
//  fft_axis_kernel  : transform along a strided axis (y or z) of a complex array [outer][rows][inner];
//                     a CTA owns 8*G adjacent columns and the whole axis.  Rows may be stored
//                     "compact": only the 2*kmax+1 modes the 2/3 rule keeps, in FFT
//                     order (0..kmax, -kmax..-1).  An inverse pass zero-fills the missing rows on
//                     load, a forward pass simply does not store them, so pruned data never
//                     touches HBM.
//  fft_x_c2r_kernel : x axis, complex half-spectrum rows -> real rows.  Two real rows share one
//                     complex transform: Z = A + iB  =>  z = a + ib.
//  fft_x_r2c_kernel : x axis, real rows -> half-spectrum rows, same pairing, split afterwards:
//                     A[k] = (Z[k] + conj Z[N-k])/2,  B[k] = (Z[k] - conj Z[N-k])/(2i).
#include "mhd_internal.h"
#include "fft_core.cuh"

#include <stdlib.h>

namespace mhd {
using namespace mhdfft;

// compact row index of full FFT index f on an axis of length n that stores nk rows (-1: not stored)
__device__ __forceinline__ int compact_index(int f, int n, int nk) {
    if (nk == n) return f;
    const int kmax = nk >> 1;
    if (f <= kmax) return f;
    if (f >= n - kmax) return f - (n - nk);
    return -1;
}

template <int N, bool INV>
__global__ void __launch_bounds__(Tile<N>::THREADS) fft_axis_kernel(AxisArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    const int tid = threadIdx.x, p = tid & 7, i = (tid >> 3) % PL::TP, g = tid / (8 * PL::TP);
    cplx* sm = reinterpret_cast<cplx*>(smraw) + (size_t)g * N * 8;
    const int col = blockIdx.x * Tile<N>::COLS + g * 8 + p;
    const bool colok = col < a.inner;
    const long long outer = (long long)blockIdx.y + (long long)blockIdx.z * gridDim.y;
    if (outer >= a.nouter) return;           // uniform per CTA
    const cplx* __restrict__ in = a.in + outer * a.in_outer + col;
    cplx* __restrict__ out = a.out + outer * a.out_outer + col;

    cplx v[PL::E];
    constexpr int R0 = PL::radix(0), RL = PL::radix(PL::NP - 1);
#pragma unroll
    for (int m = 0; m < PL::E / R0; ++m)
#pragma unroll
        for (int q = 0; q < R0; ++q) {
            const int c = compact_index(first_index<N>(i, m, q), N, a.nk_in);
            v[m * R0 + q] = (colok && c >= 0) ? in[(long long)c * a.in_row] : make_double2(0.0, 0.0);
        }
    pencil_fft<N, INV>(v, sm, i, p, tw);
    const double s = a.scale;
#pragma unroll
    for (int m = 0; m < PL::E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int c = compact_index(last_index<N>(i, m, q), N, a.nk_out);
            if (colok && c >= 0) out[(long long)c * a.out_row] = make_double2(v[m * RL + q].x * s, v[m * RL + q].y * s);
        }
}

template <int N>
__global__ void __launch_bounds__(Tile<N>::THREADS) fft_x_c2r_kernel(RowArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    const int tid = threadIdx.x, p = tid & 7, i = (tid >> 3) % PL::TP, g = tid / (8 * PL::TP);
    cplx* sm = reinterpret_cast<cplx*>(smraw) + (size_t)g * N * 8;
    const long long pen = (long long)blockIdx.x * Tile<N>::COLS + g * 8 + p;
    const long long r0 = 2 * pen;
    const bool ok = r0 < a.nrows;            // nrows is even
    const cplx* __restrict__ A = a.spec + r0 * a.spec_pitch;
    const cplx* __restrict__ B = A + a.spec_pitch;
    const int nkx = a.nkx;

    cplx v[PL::E];
    constexpr int R0 = PL::radix(0), RL = PL::radix(PL::NP - 1);
#pragma unroll
    for (int m = 0; m < PL::E / R0; ++m)
#pragma unroll
        for (int q = 0; q < R0; ++q) {
            const int k = first_index<N>(i, m, q);
            cplx z = make_double2(0.0, 0.0);
            if (ok) {
                if (k < nkx) {
                    cplx x = A[k], y = B[k];
                    if (k == 0 || 2 * k == N) { x.y = 0.0; y.y = 0.0; }   // self-conjugate modes: Im ignored
                    z = make_double2(x.x - y.y, x.y + y.x);                // A + iB
                } else if (N - k < nkx) {
                    cplx x = A[N - k], y = B[N - k];
                    z = make_double2(x.x + y.y, y.x - x.y);                // conj(A) + i conj(B)
                }
            }
            v[m * R0 + q] = z;
        }
    pencil_fft<N, true>(v, sm, i, p, tw);
    double* __restrict__ ra = a.real + r0 * a.real_pitch;
    double* __restrict__ rb = ra + a.real_pitch;
    const double s = a.scale;
    if (ok) {
#pragma unroll
        for (int m = 0; m < PL::E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int x = last_index<N>(i, m, q);
                ra[x] = v[m * RL + q].x * s;
                rb[x] = v[m * RL + q].y * s;
            }
    }
}

template <int N>
__global__ void __launch_bounds__(Tile<N>::THREADS) fft_x_r2c_kernel(RowArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    const int tid = threadIdx.x, p = tid & 7, i = (tid >> 3) % PL::TP, g = tid / (8 * PL::TP);
    cplx* sm = reinterpret_cast<cplx*>(smraw) + (size_t)g * N * 8;
    const long long pen = (long long)blockIdx.x * Tile<N>::COLS + g * 8 + p;
    const long long r0 = 2 * pen;
    const bool ok = r0 < a.nrows;
    const double* __restrict__ ra = a.real + r0 * a.real_pitch;
    const double* __restrict__ rb = ra + a.real_pitch;

    cplx v[PL::E];
    constexpr int R0 = PL::radix(0), RL = PL::radix(PL::NP - 1);
#pragma unroll
    for (int m = 0; m < PL::E / R0; ++m)
#pragma unroll
        for (int q = 0; q < R0; ++q) {
            const int x = first_index<N>(i, m, q);
            v[m * R0 + q] = ok ? make_double2(ra[x], rb[x]) : make_double2(0.0, 0.0);
        }
    pencil_fft<N, false>(v, sm, i, p, tw);
#pragma unroll
    for (int m = 0; m < PL::E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) sm[last_index<N>(i, m, q) * 8 + p] = v[m * RL + q];
    __syncthreads();
    cplx* __restrict__ A = a.spec + r0 * a.spec_pitch;
    cplx* __restrict__ B = A + a.spec_pitch;
    const double s = 0.5 * a.scale;
    if (ok) {
        for (int k = i; k < a.nkx; k += PL::TP) {
            const cplx zk = sm[k * 8 + p], zm = sm[(k == 0 ? 0 : N - k) * 8 + p];
            A[k] = make_double2((zk.x + zm.x) * s, (zk.y - zm.y) * s);
            B[k] = make_double2((zk.y + zm.y) * s, (zm.x - zk.x) * s);
        }
    }
}

// ---- launchers -----------------------------------------------------------------------------
template <int N, bool INV> static cudaError_t launch_axis_n(const AxisArgs& a, const cplx* tw, cudaStream_t st) {
    const long long outer = a.nouter;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(fft_axis_kernel<N, INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile<N>::SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const unsigned tiles = (unsigned)((a.inner + Tile<N>::COLS - 1) / Tile<N>::COLS);
    unsigned gy = (unsigned)outer, gz = 1;
    while (gy > 65535u) { gz *= 2; gy = (unsigned)((outer + gz - 1) / gz); }
    fft_axis_kernel<N, INV><<<dim3(tiles, gy, gz), Tile<N>::THREADS, Tile<N>::SMEM, st>>>(a, tw);
    count_launch();
    return cudaGetLastError();
}

template <int N> static cudaError_t launch_rows_n(bool inverse, const RowArgs& a, const cplx* tw, cudaStream_t st) {
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(fft_x_c2r_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile<N>::SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(fft_x_r2c_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile<N>::SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const long long pencils = (a.nrows + 1) / 2;
    const unsigned blocks = (unsigned)((pencils + Tile<N>::COLS - 1) / Tile<N>::COLS);
    if (inverse) fft_x_c2r_kernel<N><<<blocks, Tile<N>::THREADS, Tile<N>::SMEM, st>>>(a, tw);
    else fft_x_r2c_kernel<N><<<blocks, Tile<N>::THREADS, Tile<N>::SMEM, st>>>(a, tw);
    count_launch();
    return cudaGetLastError();
}

#define MHD_FOR_EACH_N(X) X(8) X(12) X(16) X(24) X(32) X(48) X(64) X(96) X(128) X(192) X(256) X(384) X(512) X(768) X(1024)

bool fft_size_supported(int n) {
    switch (n) {
#define X(N_) case N_:
        MHD_FOR_EACH_N(X)
#undef X
        return true;
        default: return false;
    }
}

cudaError_t launch_fft_axis(int n, bool inverse, const AxisArgs& a, const double2* tw, cudaStream_t st) {
    switch (n) {
#define X(N_) case N_: return inverse ? launch_axis_n<N_, true>(a, tw, st) : launch_axis_n<N_, false>(a, tw, st);
        MHD_FOR_EACH_N(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_fft_rows(int n, bool inverse, const RowArgs& a, const double2* tw, cudaStream_t st) {
    static const bool legacy = getenv("MHD_LEGACY_XROWS") != nullptr;
    if (!legacy && xfused_supported(n)) return launch_xrows(n, inverse, a, tw, st);   // coalesced team kernel (xfused_kernel.cu)
    switch (n) {
#define X(N_) case N_: return launch_rows_n<N_>(inverse, a, tw, st);
        MHD_FOR_EACH_N(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace mhd
