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
// V = 0: the 8 (12/24)-points-per-thread plans every kernel uses.  V = 1: "big radix" plans for the strided-axis kernels:
// 16 or 32 points per thread and only TWO passes (one shared-memory exchange instead of two), see fft_kernels.cu.
template <int N, int V = 0> struct Plan;
#define MHD_PLAN(N_, E_, NP_, R0, R1, R2, R3) MHD_PLANV(N_, 0, E_, NP_, R0, R1, R2, R3)
#define MHD_PLANV(N_, V_, E_, NP_, R0, R1, R2, R3)                                               \
    template <> struct Plan<N_, V_> {                                                            \
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
MHD_PLANV(128, 1, 16, 2, 16, 8, 1, 1)
MHD_PLANV(256, 1, 16, 2, 16, 16, 1, 1)
MHD_PLANV(512, 1, 32, 2, 32, 16, 1, 1)
MHD_PLANV(1024, 1, 32, 2, 32, 32, 1, 1)
#undef MHD_PLAN
#undef MHD_PLANV
template <int N> struct HasBigPlan { static constexpr bool value = (N == 128 || N == 256 || N == 512 || N == 1024); };

// pencil groups per CTA (8 pencils each), chosen so a CTA has 128..512 threads
template <int N, int V = 0> struct Tile {
    static constexpr int TP = Plan<N, V>::TP;
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
// ---- composite radices 16 = 4 x 4 and 32 = 4 x 8, entirely in registers, internal twiddles are compile-time constants ----
// cos / sin of 2*pi*j/32 (correctly rounded literals)
__host__ __device__ constexpr double cos32(int j) { return j == 0 ? 1.0 : j == 1 ? 0.9807852804032304 : j == 2 ? 0.9238795325112867 : j == 3 ? 0.8314696123025452 : j == 4 ? 0.7071067811865476 : j == 5 ? 0.5555702330196023 : j == 6 ? 0.38268343236508984 : j == 7 ? 0.19509032201612833 : j == 8 ? 6.123233995736766e-17 : j == 9 ? -0.1950903220161282 : j == 10 ? -0.3826834323650897 : j == 11 ? -0.555570233019602 : j == 12 ? -0.7071067811865475 : j == 13 ? -0.8314696123025453 : j == 14 ? -0.9238795325112867 : j == 15 ? -0.9807852804032304 : j == 16 ? -1.0 : j == 17 ? -0.9807852804032304 : j == 18 ? -0.9238795325112868 : j == 19 ? -0.8314696123025455 : j == 20 ? -0.7071067811865477 : j == 21 ? -0.5555702330196022 : j == 22 ? -0.38268343236509034 : j == 23 ? -0.19509032201612866 : j == 24 ? -1.8369701987210297e-16 : j == 25 ? 0.1950903220161283 : j == 26 ? 0.38268343236509 : j == 27 ? 0.5555702330196018 : j == 28 ? 0.7071067811865474 : j == 29 ? 0.8314696123025452 : j == 30 ? 0.9238795325112865 : j == 31 ? 0.9807852804032303 : 0.0; }
__host__ __device__ constexpr double sin32(int j) { return j == 0 ? 0.0 : j == 1 ? 0.19509032201612825 : j == 2 ? 0.3826834323650898 : j == 3 ? 0.5555702330196022 : j == 4 ? 0.7071067811865475 : j == 5 ? 0.8314696123025452 : j == 6 ? 0.9238795325112867 : j == 7 ? 0.9807852804032304 : j == 8 ? 1.0 : j == 9 ? 0.9807852804032304 : j == 10 ? 0.9238795325112867 : j == 11 ? 0.8314696123025455 : j == 12 ? 0.7071067811865476 : j == 13 ? 0.5555702330196022 : j == 14 ? 0.3826834323650899 : j == 15 ? 0.1950903220161286 : j == 16 ? 1.2246467991473532e-16 : j == 17 ? -0.19509032201612836 : j == 18 ? -0.38268343236508967 : j == 19 ? -0.555570233019602 : j == 20 ? -0.7071067811865475 : j == 21 ? -0.8314696123025452 : j == 22 ? -0.9238795325112865 : j == 23 ? -0.9807852804032303 : j == 24 ? -1.0 : j == 25 ? -0.9807852804032304 : j == 26 ? -0.9238795325112866 : j == 27 ? -0.8314696123025455 : j == 28 ? -0.7071067811865477 : j == 29 ? -0.5555702330196022 : j == 30 ? -0.3826834323650904 : j == 31 ? -0.19509032201612872 : 0.0; }
// a * exp(-/+ 2 pi i j / 32) for a compile-time j (forward: minus sign; inverse: plus)
template <bool INV, int J> __device__ __forceinline__ cplx mul_w32(cplx a) {
    constexpr int j = J & 31;
    if constexpr (j == 0) return a;
    else if constexpr (j == 8) return mul_mi<INV>(a);
    else if constexpr (j == 16) return make_double2(-a.x, -a.y);
    else if constexpr (j == 24) return mul_mi<!INV>(a);
    else {
        constexpr double c = cos32(j), s = INV ? sin32(j) : -sin32(j);      // w = c + i s
        return make_double2(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}
// X[k] = sum_n v[n] w_{R*S}^{nk}, n = S*n1 + n2, k = k1 + R*k2: R-point butterflies over n1 (stride S), twiddle w^{n2 k1},
// S-point butterflies over n2; the result is left in natural order.
template <bool INV> __device__ __forceinline__ void bfly16(cplx* v) {
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) bfly4<INV>(v[n2], v[4 + n2], v[8 + n2], v[12 + n2]);     // A[k1][n2] at v[4*k1 + n2]
    v[5] = mul_w32<INV, 2>(v[5]);  v[6] = mul_w32<INV, 4>(v[6]);   v[7] = mul_w32<INV, 6>(v[7]);
    v[9] = mul_w32<INV, 4>(v[9]);  v[10] = mul_w32<INV, 8>(v[10]); v[11] = mul_w32<INV, 12>(v[11]);
    v[13] = mul_w32<INV, 6>(v[13]); v[14] = mul_w32<INV, 12>(v[14]); v[15] = mul_w32<INV, 18>(v[15]);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) bfly4<INV>(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);   // X[k1 + 4*k2] at v[4*k1 + k2]
    cplx t[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) t[r] = v[r];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1)
#pragma unroll
        for (int k2 = 0; k2 < 4; ++k2) v[k1 + 4 * k2] = t[4 * k1 + k2];
}
template <bool INV, int K1> __device__ __forceinline__ void tw32_row(cplx* v) {   // v[8*K1 + n2] *= w32^(n2*K1), n2 = 1..7
    v[8 * K1 + 1] = mul_w32<INV, 1 * K1>(v[8 * K1 + 1]); v[8 * K1 + 2] = mul_w32<INV, 2 * K1>(v[8 * K1 + 2]);
    v[8 * K1 + 3] = mul_w32<INV, 3 * K1>(v[8 * K1 + 3]); v[8 * K1 + 4] = mul_w32<INV, 4 * K1>(v[8 * K1 + 4]);
    v[8 * K1 + 5] = mul_w32<INV, 5 * K1>(v[8 * K1 + 5]); v[8 * K1 + 6] = mul_w32<INV, 6 * K1>(v[8 * K1 + 6]);
    v[8 * K1 + 7] = mul_w32<INV, 7 * K1>(v[8 * K1 + 7]);
}
template <bool INV> __device__ __forceinline__ void bfly32(cplx* v) {
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) bfly4<INV>(v[n2], v[8 + n2], v[16 + n2], v[24 + n2]);    // A[k1][n2] at v[8*k1 + n2]
    tw32_row<INV, 1>(v); tw32_row<INV, 2>(v); tw32_row<INV, 3>(v);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) bfly8<INV>(&v[8 * k1]);                                   // X[k1 + 4*k2] at v[8*k1 + k2]
    cplx t[32];
#pragma unroll
    for (int r = 0; r < 32; ++r) t[r] = v[r];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1)
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) v[k1 + 4 * k2] = t[8 * k1 + k2];
}
template <int R, bool INV> __device__ __forceinline__ void bfly(cplx* v) {
    if constexpr (R == 32) bfly32<INV>(v);
    else if constexpr (R == 16) bfly16<INV>(v);
    else if constexpr (R == 8) bfly8<INV>(v);
    else if constexpr (R == 4) bfly4<INV>(v[0], v[1], v[2], v[3]);
    else if constexpr (R == 3) bfly3<INV>(v);
    else if constexpr (R == 2) bfly2<INV>(v);
}

// index of the q-th input of butterfly m held by slot i in the FIRST pass, and of the q-th output in the LAST
template <int N, int V = 0> __device__ __forceinline__ int first_index(int i, int m, int q) {
    return i + Plan<N, V>::TP * m + q * (N / Plan<N, V>::radix(0));
}
template <int N, int V = 0> __device__ __forceinline__ int last_index(int i, int m, int q) {
    return i + Plan<N, V>::TP * m + q * (N / Plan<N, V>::radix(Plan<N, V>::NP - 1));
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
template <int N, bool INV, int S, int P, typename L, int V = 0>
struct Pass {
    static constexpr int R = Plan<N, V>::radix(S);
    static constexpr int E = Plan<N, V>::E;
    static constexpr int TP = Plan<N, V>::TP;
    static constexpr bool LAST = (S == Plan<N, V>::NP - 1);
    __device__ __forceinline__ static void run(cplx (&v)[E], cplx* sm, int i, const L& lay, const cplx* __restrict__ tw) {
#pragma unroll
        for (int m = 0; m < E / R; ++m) {
            const int b = i + TP * m;
            const int k = b & (P - 1);
            if constexpr (S > 0 && V == 1) {
                // big radix: w, w^2, w^4, w^8(, w^16) from the table, every other power by ONE multiplication chain of depth <= 3
                // (15 or 31 table reads per butterfly would cost more load-store wavefronts than the exchange they replace)
                cplx w[R];
#pragma unroll
                for (int q = 1; q < R; q <<= 1) {
                    w[q] = __ldg(&tw[k * q * (N / (P * R))]);
                    if (INV) w[q].y = -w[q].y;
                }
#pragma unroll
                for (int q = 3; q < R; ++q)
                    if ((q & (q - 1)) != 0) w[q] = cmul(w[q & (q - 1)], w[q & -q]);      // q = (q without its lowest bit) + lowest bit
#pragma unroll
                for (int q = 1; q < R; ++q) v[m * R + q] = cmul(v[m * R + q], w[q]);
            } else if constexpr (S > 0) {
#pragma unroll
                for (int q = 1; q < R; ++q) {
                    cplx w = __ldg(&tw[k * q * (N / (P * R))]);
                    if (INV) w.y = -w.y;
                    v[m * R + q] = cmul(v[m * R + q], w);
                }
            }
            bfly<R, INV>(&v[m * R]);
            if constexpr (!LAST) {
                const int j = (b - k) * R + k;
#pragma unroll
                for (int q = 0; q < R; ++q) sm[lay(j + q * P)] = v[m * R + q];
            }
        }
        if constexpr (!LAST) {
            constexpr int Rn = Plan<N, V>::radix(S + 1);
            __syncthreads();
#pragma unroll
            for (int m = 0; m < E / Rn; ++m)
#pragma unroll
                for (int q = 0; q < Rn; ++q) v[m * Rn + q] = sm[lay(i + TP * m + q * (N / Rn))];
            __syncthreads();
            Pass<N, INV, S + 1, P * R, L, V>::run(v, sm, i, lay, tw);
        }
    }
};

// Transform the pencil whose first-pass inputs are in v (see first_index); on return v holds the
// last-pass outputs (see last_index).  All threads of the CTA must call it (it synchronises).
template <int N, bool INV, int V = 0>
__device__ __forceinline__ void pencil_fft(cplx (&v)[Plan<N, V>::E], cplx* sm, int i, int p, const cplx* __restrict__ tw) {
    Cols8 lay{p};
    Pass<N, INV, 0, 1, Cols8, V>::run(v, sm, i, lay, tw);
}
// same for 4 pencils side by side (lane = (p = tid & 3, slot))
template <int N, bool INV>
__device__ __forceinline__ void pencil_fft4(cplx (&v)[Plan<N>::E], cplx* sm, int i, int p, const cplx* __restrict__ tw) {
    Cols4 lay{p};
    Pass<N, INV, 0, 1, Cols4>::run(v, sm, i, lay, tw);
}
// same, one pencil per (padded) buffer
template <int N, bool INV>
__device__ __forceinline__ void pencil_fft_private(cplx (&v)[Plan<N>::E], cplx* sm, int i, const cplx* __restrict__ tw) {
    Padded lay;
    Pass<N, INV, 0, 1, Padded>::run(v, sm, i, lay, tw);
}

}  // namespace mhdfft
