// peaks_kernel.cu — measured ceilings of the two on-chip resources that bound the fused x pass (instrumentation, not on the
// solver's path): the FP64 FMA pipe and the shared-memory data path, and what the fused pass's own exchange pattern reaches.  SURVEY.md §8(d) leaves the FP64 peak "nominal —
// builder to measure"; bench.py --workload peaks (and the default bench line) report x_fused against these numbers.
//
//   fp64 : every thread runs 8 independent DFMA chains (x = x*a + b), 148*k CTAs of 256 threads, no memory traffic.
//          flops = 2 per DFMA.
//   smem : every thread alternates conflict-free STS.128 / LDS.128 on its own 16-byte slot pattern (a warp moves 512 B =
//          4 wavefronts of 128 B per instruction).  bytes = 16 per thread per instruction.
#include "mhd_internal.h"

namespace mhd {

__global__ void __launch_bounds__(256) peak_fp64_kernel(double* __restrict__ out, int iters, double a, double b) {
    double x0 = threadIdx.x * 1e-3, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0, x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

__global__ void __launch_bounds__(256) peak_smem_kernel(double* __restrict__ out, int iters) {
    __shared__ double2 sm[4 * 256];
    double2 v0 = make_double2(threadIdx.x, 1.0), v1 = make_double2(2.0, threadIdx.x), v2 = v0, v3 = v1;
    double2* p = sm + threadIdx.x;              // consecutive lanes -> consecutive 16-byte slots: conflict-free
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        p[0] = v0; p[256] = v1; p[512] = v2; p[768] = v3;
        __syncwarp();
        const int o = (it & 1) ? 1 : 31;        // read a neighbour's slot of the same warp so nothing is forwarded in registers
        const double2* q = sm + (threadIdx.x & ~31) + ((threadIdx.x + o) & 31);
        v0 = q[0]; v1 = q[256]; v2 = q[512]; v3 = q[768];
        __syncwarp();
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = v0.x + v1.y + v2.x + v3.y;
}

// exchange: the fused x pass's own pattern with everything else stripped away.  One persistent CTA of 256 threads per SM,
//          4 teams of 64 threads; per iteration a thread holds two sets of 8 complex values, runs DFMA_PER_ITER dependent-free
//          DFMAs on them, and exchanges both sets through team-private padded buffers (barrier, 16 STS.128 with the first-pass
//          index set, barrier, 16 LDS.128 with the stride-64 index set; see MODE): what the 8 warps of an SM can pull through the
//          load-store pipe when the traffic comes in barrier-synchronised bursts with FP64 work in between.
//          bytes = 32 x 16 per thread per iteration.
#define MHD_PAD8(e) ((e) + ((e) >> 3))
// MODE 0: write, barrier, read, barrier; 1: barrier, write, barrier, read (the shipped x passes); 2: two buffers per set used
// alternately, ONE barrier per exchange (write, barrier, read); 3: no shared memory and no barrier at all -- the same 16 complex
// values per thread are exchanged by an 8 x 8 register transpose among the 8 lanes of a warp octet (three __shfl_xor_sync
// butterfly rounds, 4 of the 8 values of a set per round): the most a warp-shuffle exchange could do for a radix-8 pass, as
// an upper bound for the north-star's "warp-shuffle butterflies" question (a 64-thread team would still need one
// shared-memory exchange on top, because its transposition spans two warps)
__device__ __forceinline__ double2 shfl_xor_c(double2 x, int mask) {
    x.x = __shfl_xor_sync(0xffffffffu, x.x, mask);
    x.y = __shfl_xor_sync(0xffffffffu, x.y, mask);
    return x;
}
// one butterfly round of the octet transpose: lanes whose bit R is 0 give away the values whose index has bit R set, and v.v.
template <int R> __device__ __forceinline__ void transpose_round(double2 (&v)[8], bool hi) {
#pragma unroll
    for (int q0 = 0; q0 < 8; ++q0) {
        if (q0 & (1 << R)) continue;
        const int q1 = q0 | (1 << R);
        const double2 send = hi ? v[q0] : v[q1];
        const double2 recv = shfl_xor_c(send, 1 << R);
        if (hi) v[q0] = recv; else v[q1] = recv;
    }
}
template <int REPS, int MODE>
__global__ void __launch_bounds__(256, 1) peak_exchange_kernel(double* __restrict__ out, int iters, double a, double b) {
    extern __shared__ __align__(16) unsigned char smraw[];
    const int team = threadIdx.x / 64, i = threadIdx.x % 64;
    double2* const base = reinterpret_cast<double2*>(smraw) + (size_t)team * 4 * 640;
    double2 v[8], w[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { v[q] = make_double2(i + q, q); w[q] = make_double2(q, i); }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < REPS; ++r)
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                v[q].x = fma(v[q].x, a, b); v[q].y = fma(v[q].y, a, -b);
                w[q].x = fma(w[q].x, a, b); w[q].y = fma(w[q].y, a, -b);
            }
        if (MODE == 3) {
            const int lane = threadIdx.x & 31;
            transpose_round<0>(v, lane & 1); transpose_round<0>(w, lane & 1);
            transpose_round<1>(v, lane & 2); transpose_round<1>(w, lane & 2);
            transpose_round<2>(v, lane & 4); transpose_round<2>(w, lane & 4);
            continue;
        }
        double2* const A = base + ((MODE == 2) ? (it & 1) * 1280 : 0);
        double2* const B = A + 640;
        if (MODE == 1) asm volatile("bar.sync %0, 64;" ::"r"(team + 1) : "memory");
#pragma unroll
        for (int q = 0; q < 8; ++q) { A[MHD_PAD8(i * 8 + q)] = v[q]; B[MHD_PAD8(i * 8 + q)] = w[q]; }
        asm volatile("bar.sync %0, 64;" ::"r"(team + 1) : "memory");
#pragma unroll
        for (int q = 0; q < 8; ++q) { v[q] = A[MHD_PAD8(i + 64 * q)]; w[q] = B[MHD_PAD8(i + 64 * q)]; }
        if (MODE == 0) asm volatile("bar.sync %0, 64;" ::"r"(team + 1) : "memory");
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += (v[q].x + v[q].y) + (w[q].x + w[q].y);
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Achieved shared-memory GB/s of the exchange pattern above with 32*REPS DFMAs per thread between exchanges (REPS = 6 is the
// fused x pass's ratio at N = 512: ~190 FP64 instructions per thread and transform pass).  scratch: >= sms*256 doubles.
cudaError_t measure_exchange(double* scratch, size_t scratch_doubles, cudaStream_t st, int dfma_per_exchange, int mode, double* smem_gbs) {
    const int dev = device_slot();
    int sms = 0;
    cudaError_t e = device_sm_count(dev, &sms);
    if (e != cudaSuccess) return e;
    if (scratch_doubles < (size_t)sms * 256) return cudaErrorInvalidValue;
    const int reps = dfma_per_exchange / 32;
    void (*kern)(double*, int, double, double) = nullptr;
#define MHD_EXCH(R_)                                                                              \
    case R_: kern = mode == 0 ? peak_exchange_kernel<R_, 0> : mode == 1 ? peak_exchange_kernel<R_, 1> : mode == 2 ? peak_exchange_kernel<R_, 2> : peak_exchange_kernel<R_, 3>; break;
    if (mode < 0 || mode > 3) return cudaErrorInvalidValue;
    switch (reps) {
        MHD_EXCH(0) MHD_EXCH(2) MHD_EXCH(4) MHD_EXCH(6) MHD_EXCH(8)
        default: return cudaErrorInvalidValue;
    }
#undef MHD_EXCH
    const int smem = 4 * 4 * 640 * (int)sizeof(double2);
    if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    cudaEvent_t a, b;
    if ((e = cudaEventCreate(&a)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&b)) != cudaSuccess) { cudaEventDestroy(a); return e; }
    double best = 0.0;
    const int iters = 8192;
    for (int r = 0; r < 4 && e == cudaSuccess; ++r) {
        cudaEventRecord(a, st);
        kern<<<sms, 256, smem, st>>>(scratch, iters, 0.999999, 1e-9);
        count_launch();
        cudaEventRecord(b, st);
        if ((e = cudaEventSynchronize(b)) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        const double bytes = 32.0 * 16.0 * (double)iters * 256.0 * (double)sms;
        if (r > 0 && ms > 0.f) best = fmax(best, bytes / (ms * 1e-3) / 1e9);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (e == cudaSuccess) e = cudaGetLastError();
    *smem_gbs = best;
    return e;
}

// scratch: >= grid*256 doubles.  Best of `reps` launches each; results in TFLOP/s and GB/s.
cudaError_t measure_peaks(double* scratch, size_t scratch_doubles, cudaStream_t st, double* fp64_tflops, double* smem_gbs) {
    const int dev = device_slot();
    int sms = 0;
    cudaError_t e = device_sm_count(dev, &sms);
    if (e != cudaSuccess) return e;
    const int grid = sms * 8;                   // 8 CTAs of 256 threads per SM: 64 warps per SM
    if (scratch_doubles < (size_t)grid * 256) return cudaErrorInvalidValue;
    cudaEvent_t a, b;
    if ((e = cudaEventCreate(&a)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&b)) != cudaSuccess) { cudaEventDestroy(a); return e; }
    const int reps = 5;
    double best_f = 0.0, best_s = 0.0;
    for (int r = 0; r < reps + 1 && e == cudaSuccess; ++r) {
        const int iters = 4096;
        cudaEventRecord(a, st);
        peak_fp64_kernel<<<grid, 256, 0, st>>>(scratch, iters, 0.999999, 1e-9);
        count_launch();
        cudaEventRecord(b, st);
        if ((e = cudaEventSynchronize(b)) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        const double flops = 2.0 * 8.0 * 16.0 * (double)iters * 256.0 * (double)grid;
        if (r > 0 && ms > 0.f) best_f = fmax(best_f, flops / (ms * 1e-3) / 1e12);
        const int it2 = 8192;
        cudaEventRecord(a, st);
        peak_smem_kernel<<<grid, 256, 0, st>>>(scratch, it2);
        count_launch();
        cudaEventRecord(b, st);
        if ((e = cudaEventSynchronize(b)) != cudaSuccess) break;
        cudaEventElapsedTime(&ms, a, b);
        const double bytes = 16.0 * 8.0 * (double)it2 * 256.0 * (double)grid;      // 4 stores + 4 loads of 16 B per iteration
        if (r > 0 && ms > 0.f) best_s = fmax(best_s, bytes / (ms * 1e-3) / 1e9);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (e == cudaSuccess) e = cudaGetLastError();
    *fp64_tflops = best_f;
    *smem_gbs = best_s;
    return e;
}

}  // namespace mhd
