// fft_kernels.cu — batched pencil-FFT kernels for sm_100a (fp64), built on fft_core.cuh.
//
//  fft_axis_kernel  : transform along a strided axis (y or z) of a complex array [outer][rows][inner];
//                     a CTA owns 8*G adjacent columns and the whole axis.  Rows may be stored
//                     "compact": only the 2*kmax+1 modes the 2/3 rule keeps, in FFT
//                     order (0..kmax, -kmax..-1).  An inverse pass zero-fills the missing rows on
//                     load, a forward pass simply does not store them, so pruned data never
//                     touches HBM.
//  The x axis (real rows <-> half-spectrum rows, two real rows per complex transform) lives in xfused_kernel.cu.
//
//  Measured and not kept (round 2, 512^3, profiles/r02_experiments.md): 32 points per thread with a single exchange (slower:
//  168 registers, 12 warps/SM), TMA / cp.async staging of the next tile in a persistent CTA (slower: one CTA per SM), a
//  persistent tile loop with L2 prefetch (slower than letting the hardware scheduler start a fresh CTA per tile).  With the
//  transform removed this access pattern runs at 0.85-1.0 of the copy bandwidth; with it, at 0.70-0.83.
#include "mhd_internal.h"
#include "fft_core.cuh"

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

// exchange synchronisation of the strided-axis kernels (fft_core.cuh Pass<..., SYNC>): every CTA transforms ONE tile and exits,
// so the barrier after the last exchange's reads protects nothing (1); 2 = two buffers, one barrier per exchange
#ifndef MHD_AXIS_SYNC
#define MHD_AXIS_SYNC 1
#endif
#ifndef MHD_AXIS24_MINB
#define MHD_AXIS24_MINB 2     // minimum CTAs per SM asked of ptxas for the 24-points-per-thread lengths (0: no request)
#endif
template <int N, bool INV>
__global__ void __launch_bounds__(Tile<N>::THREADS, (Plan<N>::E == 24 ? MHD_AXIS24_MINB : 0)) fft_axis_kernel(AxisArgs a, const cplx* __restrict__ tw) {
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
    pencil_fft<N, INV, (MHD_AXIS_SYNC == 2 ? 1 : MHD_AXIS_SYNC)>(v, sm, i, p, tw);      // (two buffers only in the 4-column variant)
    const double s = a.scale;
#pragma unroll
    for (int m = 0; m < PL::E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int c = compact_index(last_index<N>(i, m, q), N, a.nk_out);
            if (colok && c >= 0) out[(long long)c * a.out_row] = make_double2(v[m * RL + q].x * s, v[m * RL + q].y * s);
        }
}

// Variant measured in round 3 (profiles/r03_experiments.md): 4 adjacent columns per CTA instead of 8, so a 512-long axis runs
// in 256-thread CTAs, four per SM, and a __syncthreads stalls 8 warps instead of 16 (64-byte row segments in HBM instead of
// 128).  Compile-time switch: -DMHD_AXIS_COLS4_MIN=<smallest N that uses it>; 0 (default) = never.
#ifndef MHD_AXIS_COLS4_MIN
#define MHD_AXIS_COLS4_MIN 0
#endif
template <int N, bool INV>
__global__ void __launch_bounds__(Plan<N>::TP * 4) fft_axis4_kernel(AxisArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    const int tid = threadIdx.x, p = tid & 3, i = tid >> 2;
    cplx* sm = reinterpret_cast<cplx*>(smraw);
    const int col = blockIdx.x * 4 + p;
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
    pencil_fft4<N, INV, MHD_AXIS_SYNC>(v, sm, i, p, tw);
    const double s = a.scale;
#pragma unroll
    for (int m = 0; m < PL::E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int c = compact_index(last_index<N>(i, m, q), N, a.nk_out);
            if (colok && c >= 0) out[(long long)c * a.out_row] = make_double2(v[m * RL + q].x * s, v[m * RL + q].y * s);
        }
}

// ---- launchers -----------------------------------------------------------------------------
template <int N, bool INV> static cudaError_t launch_axis_n(const AxisArgs& a, const cplx* tw, cudaStream_t st) {
    const long long outer = a.nouter;
    static DeviceOnce once;
    const int dev = device_slot();
    if (dev < 0) return cudaErrorInvalidDevice;
    if (!once.done[dev]) {
        cudaError_t e = cudaFuncSetAttribute(fft_axis_kernel<N, INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile<N>::SMEM);
        if (e != cudaSuccess) return e;
        once.done[dev] = true;
    }
    unsigned gy = (unsigned)outer, gz = 1;
    while (gy > 65535u) { gz *= 2; gy = (unsigned)((outer + gz - 1) / gz); }
    if constexpr (MHD_AXIS_COLS4_MIN > 0 && N >= MHD_AXIS_COLS4_MIN && Plan<N>::E == 8 && Plan<N>::TP * 4 >= 64) {
        static DeviceOnce once4;
        constexpr int smem4 = N * 4 * (int)sizeof(cplx) * (MHD_AXIS_SYNC == 2 ? 2 : 1);
        if (!once4.done[dev]) {
            cudaError_t e = cudaFuncSetAttribute(fft_axis4_kernel<N, INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem4);
            if (e != cudaSuccess) return e;
            once4.done[dev] = true;
        }
        fft_axis4_kernel<N, INV><<<dim3((unsigned)((a.inner + 3) / 4), gy, gz), Plan<N>::TP * 4, smem4, st>>>(a, tw);
        count_launch();
        return cudaGetLastError();
    }
    const unsigned tiles = (unsigned)((a.inner + Tile<N>::COLS - 1) / Tile<N>::COLS);
    fft_axis_kernel<N, INV><<<dim3(tiles, gy, gz), Tile<N>::THREADS, Tile<N>::SMEM, st>>>(a, tw);
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
    return launch_xrows(n, inverse, a, tw, st);   // coalesced team kernels (xfused_kernel.cu), every supported length
}

}  // namespace mhd
