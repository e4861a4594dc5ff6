// fft_core.cuh — in-register / shared-memory Stockham pencil FFT for sm_100a, fp64.
//
// One "pencil" is a 1-D complex transform of compile-time length N (the FFT under the
// pseudo-spectral derivative; the paper calls cuFFT/AccFFT, here it is hand-written).  Eight pencils
// that are adjacent in memory are transformed side by side: lane = (pencil p = tid & 7,
// slot i = tid >> 3).  A warp therefore touches 4 rows x 8 pencils x 16 B = four full 128-byte
// lines in global memory and four conflict-free wavefronts in shared memory, for any stride.
//
// Each thread keeps E = N/TP elements in registers.  A pass of radix r does E/r butterflies per
// thread; between passes the data is exchanged through one shared buffer laid out [N][8] complex.
// Stockham auto-sort indexing (P = product of the radices already done, t = N/r):
//     butterfly b:  k = b mod P,  inputs x[b + q*t],  twiddle w_N^(k*q*N/(P*r)),  outputs y[(b-k)*r + k + q*P]
// so the first pass reads rows b + q*N/r0 and the last pass leaves X[b + q*N/rL] in registers,
// which lets the callers load from and store to global memory directly, with no extra staging.
#pragma once
#include <cuda_runtime.h>

#ifndef MHD_AXIS_TWCHAIN
// twiddles of a radix-4/8 pass of the strided-axis kernels: 1 = w from the table, w^2..w^7 by multiplication; 0 = all from the table
#define MHD_AXIS_TWCHAIN 1
#endif

namespace mhdfft {

typedef double2 cplx;

__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
// a * (-i) for the forward transform, a * (+i) for the inverse
template <bool INV>
__device__ __forceinline__ cplx mul_mi(cplx a) {
    return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}

// ---- radix plans ---------------------------------------------------------------------------
// radices in execution order; a factor 3, if any, goes last so that P stays a power of two.
template <int N> struct Plan;
#define MHD_PLAN(N_, E_, NP_, R0, R1, R2, R3)                                                    \
    template <> struct Plan<N_> {                                                                \
        static constexpr int E = E_;   /* elements per thread */                                 \
        static constexpr int NP = NP_; /* passes */                                              \
        static constexpr int TP = N_ / E_; /* threads per pencil */                              \
        __host__ __device__ static constexpr int radix(int s) {                                  \
            return s == 0 ? R0 : s == 1 ? R1 : s == 2 ? R2 : R3;                                 \
        }                                                                                        \
    };
MHD_PLAN(8, 8, 1, 8, 1, 1, 1)
MHD_PLAN(16, 8, 2, 8, 2, 1, 1)
MHD_PLAN(32, 8, 2, 8, 4, 1, 1)
MHD_PLAN(64, 8, 2, 8, 8, 1, 1)
MHD_PLAN(128, 8, 3, 8, 4, 4, 1)
MHD_PLAN(256, 8, 3, 8, 8, 4, 1)
MHD_PLAN(512, 8, 3, 8, 8, 8, 1)
MHD_PLAN(1024, 8, 4, 8, 8, 4, 4)
MHD_PLAN(12, 12, 2, 4, 3, 1, 1)
MHD_PLAN(24, 24, 2, 8, 3, 1, 1)
MHD_PLAN(48, 12, 3, 4, 4, 3, 1)
MHD_PLAN(96, 24, 3, 8, 4, 3, 1)
MHD_PLAN(192, 24, 3, 8, 8, 3, 1)
MHD_PLAN(384, 24, 4, 8, 4, 4, 3)
MHD_PLAN(768, 24, 4, 8, 8, 4, 3)
#undef MHD_PLAN

// pencil groups per CTA (8 pencils each), chosen so a CTA has 128..512 threads
template <int N> struct Tile {
    static constexpr int TP = Plan<N>::TP;
    static constexpr int G = (8 * TP >= 128) ? 1 : 128 / (8 * TP);
    static constexpr int THREADS = 8 * TP * G;
    static constexpr int COLS = 8 * G;                       // pencils per CTA
    static constexpr size_t SMEM = (size_t)N * COLS * sizeof(cplx);
};

// ---- butterflies (natural-order outputs) ---------------------------------------------------
template <bool INV> __device__ __forceinline__ void bfly2(cplx* v) {
    cplx a = v[0], b = v[1];
    v[0] = cadd(a, b); v[1] = csub(a, b);
}
template <bool INV> __device__ __forceinline__ void bfly4(cplx& a0, cplx& a1, cplx& a2, cplx& a3) {
    cplx t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_mi<INV>(csub(a1, a3));
    a0 = cadd(t0, t2); a1 = cadd(t1, t3); a2 = csub(t0, t2); a3 = csub(t1, t3);
}
template <bool INV> __device__ __forceinline__ void bfly3(cplx* v) {
    const double h = 0.86602540378443864676;  // sqrt(3)/2
    cplx t = cadd(v[1], v[2]), d = csub(v[1], v[2]);
    cplx m = make_double2(v[0].x - 0.5 * t.x, v[0].y - 0.5 * t.y);
    cplx s = mul_mi<INV>(make_double2(h * d.x, h * d.y));   // (-/+ i) * sqrt(3)/2 * (v1 - v2)
    v[0] = cadd(v[0], t); v[1] = cadd(m, s); v[2] = csub(m, s);
}
template <bool INV> __device__ __forceinline__ void bfly8(cplx* v) {
    const double r = 0.70710678118654752440;  // 1/sqrt(2)
    cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    cplx o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
    bfly4<INV>(e0, e1, e2, e3);
    bfly4<INV>(o0, o1, o2, o3);
    // o_k *= w8^k, w8 = exp(-/+ i pi/4)
    cplx w1 = INV ? make_double2(r * (o1.x - o1.y), r * (o1.x + o1.y)) : make_double2(r * (o1.x + o1.y), r * (o1.y - o1.x));
    cplx w2 = mul_mi<INV>(o2);
    cplx w3 = INV ? make_double2(r * (-o3.x - o3.y), r * (o3.x - o3.y)) : make_double2(r * (o3.y - o3.x), r * (-o3.x - o3.y));
    v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
    v[1] = cadd(e1, w1); v[5] = csub(e1, w1);
    v[2] = cadd(e2, w2); v[6] = csub(e2, w2);
    v[3] = cadd(e3, w3); v[7] = csub(e3, w3);
}
template <int R, bool INV> __device__ __forceinline__ void bfly(cplx* v) {
    if constexpr (R == 8) bfly8<INV>(v);
    else if constexpr (R == 4) bfly4<INV>(v[0], v[1], v[2], v[3]);
    else if constexpr (R == 3) bfly3<INV>(v);
    else if constexpr (R == 2) bfly2<INV>(v);
}

// index of the q-th input of butterfly m held by slot i in the FIRST pass, and of the q-th output in the LAST
template <int N> __device__ __forceinline__ int first_index(int i, int m, int q) {
    return i + Plan<N>::TP * m + q * (N / Plan<N>::radix(0));
}
template <int N> __device__ __forceinline__ int last_index(int i, int m, int q) {
    return i + Plan<N>::TP * m + q * (N / Plan<N>::radix(Plan<N>::NP - 1));
}
// position in the register array of (butterfly m, leg q) for first / last pass
template <int N> __device__ __forceinline__ constexpr int first_reg(int m, int q) { return m * Plan<N>::radix(0) + q; }
template <int N> __device__ __forceinline__ constexpr int last_reg(int m, int q) { return m * Plan<N>::radix(Plan<N>::NP - 1) + q; }

// ---- shared-memory layouts of one exchange buffer ------------------------------------------------
// Cols8 : [N][8] complex, element e of pencil p at e*8 + p.  With lane = (p, slot) any set of rows is
//         conflict-free (each row is one full 128-byte wavefront), whatever the stride between rows.
// Padded: one pencil per buffer, element e at e + (e >> 3) (one pad slot per 8 elements).  With lanes
//         = consecutive slots of ONE pencil this keeps the stride-8 / stride-64 writes of the
//         radix-8 passes on distinct 16-byte bank groups.
struct Cols8 {
    int p;
    __device__ __forceinline__ int operator()(int e) const { return e * 8 + p; }
};
// Cols4 : [N][4] complex, 64 bytes per element row.  A quarter-warp (4 pencils x 2 adjacent slots) touches two rows; they
//         must fall on opposite halves of the 128-byte bank period, so the row index has its lowest bit flipped by the
//         parity of bits 3 and 6 (adjacent slots differ in bit 0 on reads / radix-8 second-pass writes, in bit 3 on
//         first-pass writes).
struct Cols4 {
    int p;
    __device__ __forceinline__ int operator()(int e) const { return ((e ^ (((e >> 3) ^ (e >> 6)) & 1)) << 2) + p; }
};
struct Padded {
    __device__ __forceinline__ int operator()(int e) const { return e + (e >> 3); }
    __host__ __device__ static constexpr int size(int n) { return n + (n >> 3) + 1; }
};

// ---- the passes ----------------------------------------------------------------------------
// tw[j] = exp(-2*pi*i*j/N), j = 0..N-1 (forward); the inverse conjugates on the fly.
// sm + lay(e): where element e of this thread's pencil lives between passes.  i: slot (0..TP-1).
// SYNC: how the exchange between two passes is synchronised.
//   0  write, barrier, read, barrier -- always safe: the caller may write the buffer again right after run() returns (loops)
//   1  the same, without the barrier after the LAST exchange's reads: for callers that never touch the buffer again
//      (one pencil tile per CTA), one barrier fewer per transform
//   2  two buffers used alternately (exchange S in buffer S & 1, BUF complex apart), one barrier per exchange: the barrier
//      of exchange S+1 already orders every read of exchange S before the writes of exchange S+2 into the same buffer
template <int N, bool INV, int S, int P, typename L, int SYNC = 0, int BUF = 0>
struct Pass {
    static constexpr int R = Plan<N>::radix(S);
    static constexpr int E = Plan<N>::E;
    static constexpr int TP = Plan<N>::TP;
    static constexpr bool LAST = (S == Plan<N>::NP - 1);
    __device__ __forceinline__ static void run(cplx (&v)[E], cplx* sm, int i, const L& lay, const cplx* __restrict__ tw) {
#pragma unroll
        for (int m = 0; m < E / R; ++m) {
            const int b = i + TP * m;
            const int k = b & (P - 1);
            if constexpr (S > 0) {
                if constexpr (MHD_AXIS_TWCHAIN && (R == 8 || R == 4)) {
                    // one table read per butterfly, the other powers by multiplication (depth <= 3, a few ulp): the strided-axis
                    // kernels are co-limited by the load-store pipe, and 7 twiddle reads per butterfly were 18 % of its wavefronts
                    cplx w1 = __ldg(&tw[k * (N / (P * R))]);
                    if (INV) w1.y = -w1.y;
                    const cplx w2 = cmul(w1, w1), w3 = cmul(w2, w1);
                    v[m * R + 1] = cmul(v[m * R + 1], w1); v[m * R + 2] = cmul(v[m * R + 2], w2); v[m * R + 3] = cmul(v[m * R + 3], w3);
                    if constexpr (R == 8) {
                        const cplx w4 = cmul(w2, w2), w5 = cmul(w4, w1), w6 = cmul(w3, w3), w7 = cmul(w4, w3);
                        v[m * R + 4] = cmul(v[m * R + 4], w4); v[m * R + 5] = cmul(v[m * R + 5], w5);
                        v[m * R + 6] = cmul(v[m * R + 6], w6); v[m * R + 7] = cmul(v[m * R + 7], w7);
                    }
                } else {
#pragma unroll
                    for (int q = 1; q < R; ++q) {
                        cplx w = __ldg(&tw[k * q * (N / (P * R))]);
                        if (INV) w.y = -w.y;
                        v[m * R + q] = cmul(v[m * R + q], w);
                    }
                }
            }
            bfly<R, INV>(&v[m * R]);
            if constexpr (!LAST) {
                const int j = (b - k) * R + k;
                cplx* buf = sm + ((SYNC == 2 && (S & 1)) ? BUF : 0);
#pragma unroll
                for (int q = 0; q < R; ++q) buf[lay(j + q * P)] = v[m * R + q];
            }
        }
        if constexpr (!LAST) {
            constexpr int Rn = Plan<N>::radix(S + 1);
            const cplx* buf = sm + ((SYNC == 2 && (S & 1)) ? BUF : 0);
            __syncthreads();
#pragma unroll
            for (int m = 0; m < E / Rn; ++m)
#pragma unroll
                for (int q = 0; q < Rn; ++q) v[m * Rn + q] = buf[lay(i + TP * m + q * (N / Rn))];
            constexpr bool next_is_last = (S + 1 == Plan<N>::NP - 1);
            if constexpr (SYNC == 0 || (SYNC == 1 && !next_is_last)) __syncthreads();
            Pass<N, INV, S + 1, P * R, L, SYNC, BUF>::run(v, sm, i, lay, tw);
        }
    }
};

// Transform the pencil whose first-pass inputs are in v (see first_index); on return v holds the
// last-pass outputs (see last_index).  All threads of the CTA must call it (it synchronises).
template <int N, bool INV, int SYNC = 0>
__device__ __forceinline__ void pencil_fft(cplx (&v)[Plan<N>::E], cplx* sm, int i, int p, const cplx* __restrict__ tw) {
    Cols8 lay{p};
    Pass<N, INV, 0, 1, Cols8, SYNC, N * 8>::run(v, sm, i, lay, tw);
}
// same for 4 pencils side by side (lane = (p = tid & 3, slot))
template <int N, bool INV, int SYNC = 0>
__device__ __forceinline__ void pencil_fft4(cplx (&v)[Plan<N>::E], cplx* sm, int i, int p, const cplx* __restrict__ tw) {
    Cols4 lay{p};
    Pass<N, INV, 0, 1, Cols4, SYNC, N * 4>::run(v, sm, i, lay, tw);
}
// same, one pencil per (padded) buffer
template <int N, bool INV>
__device__ __forceinline__ void pencil_fft_private(cplx (&v)[Plan<N>::E], cplx* sm, int i, const cplx* __restrict__ tw) {
    Padded lay;
    Pass<N, INV, 0, 1, Padded>::run(v, sm, i, lay, tw);
}

}  // namespace mhdfft
