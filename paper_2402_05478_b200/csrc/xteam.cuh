// xteam.cuh — the "team" Stockham passes shared by the x-axis kernels (xfused_kernel.cu, planefft_kernel.cu):
// a TEAM of TP = N/E threads owns one complex transform of compile-time length N; lane = slot i, consecutive lanes hold
// consecutive elements, so global rows are read and written as full lines.  Between passes the data goes through a
// team-private padded shared buffer (element e at e + e/8: the stride-8 / stride-64 writes of the radix-8 passes fall on
// distinct 16-byte bank groups); teams synchronise among themselves only (named barrier, or __syncwarp when a team fits
// a warp).  Twiddles come from per-pass shared tables laid out [leg][k].
#pragma once
#include "fft_core.cuh"

#ifndef MHD_XF_TWCHAIN
// twiddles w^2..w^7 of a radix-8 pass by multiplication from w: 0 = never (7 table reads), 1 = passes with P >= 32 only,
// 2 = every pass, 3 = table reads while the table row is one broadcast wavefront (P < 32), else w, w^2, w^4 + 4 products.
#define MHD_XF_TWCHAIN 2
#endif
// the same choice for the two-transform passes (XPass2), where one set of twiddles serves both transforms
#ifndef MHD_XF2_TW
#define MHD_XF2_TW 2
#endif

#ifndef MHD_XF2_TWREG
// 1: the thread's own w of every radix-8 pass lives in registers for the whole kernel (4 doubles at N = 512) instead of
// being re-read from the shared table by every transform pair
#define MHD_XF2_TWREG 1
#endif
#ifndef MHD_XF2_LATEBAR
// XPass2 barrier placement: 0 = write, barrier, read, barrier (the buffers are free again as soon as a pass returns);
// 1 = barrier, write, barrier, read: the "reads are done" barrier moves in front of the NEXT write, so the reads of an
// exchange and the twiddle chain / butterflies that consume them are one scheduling region.  Callers then synchronise the
// team before they write the exchange buffers themselves.  2 = the same, and transform A's writes are issued before
// transform B's butterflies of the pass, so the load-store pipe drains them under arithmetic.
// Measured at 512^3 (x_fused, ms): 0: 4.84, 1: 4.76, 2: 4.73 in one session (profiles/r02_experiments.md).
#define MHD_XF2_LATEBAR 2
#endif

namespace mhd {
using namespace mhdfft;

template <int N> struct XCfg {
    static constexpr int TP = Plan<N>::TP;                      // threads per row
    static constexpr int BUF = Padded::size(N);                 // complex elements per exchange buffer
    // number of twiddle-table entries: sum over passes s >= 1 of (R_s - 1) * P_s
    __host__ __device__ static constexpr int tw_offset(int s) {  // first entry of pass s
        int off = 0, P = Plan<N>::radix(0);
        for (int t = 1; t < s; ++t) { off += (Plan<N>::radix(t) - 1) * P; P *= Plan<N>::radix(t); }
        return off;
    }
    static constexpr int NTW = tw_offset(Plan<N>::NP);
};

template <int TP> __device__ __forceinline__ void team_sync(int team) {
    if constexpr (TP >= 64) asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(TP) : "memory");
    else __syncwarp();
}

__device__ __forceinline__ constexpr int xpad(int e) { return e + (e >> 3); }
// padded index of (e + D) for a compile-time D, given e and xpad(e)
template <int D> __device__ __forceinline__ int xpad_add(int e, int pe) {
    if constexpr (D % 8 == 0) return pe + D + D / 8;
    else return xpad(e + D);
}

// One Stockham pass S (P = product of the radices done) on the 8 register values of slot i; the
// exchange before the next pass goes through sm0 (the following one through sm1, and so on).
// SINGLE: sm0 == sm1 (one buffer per team): a second team barrier after the reads protects the next pass's writes.
template <int N, bool INV, int S, int P, bool SINGLE = false>
struct XPass {
    using PL = Plan<N>;
    static constexpr int R = PL::radix(S);
    static constexpr int E = PL::E;
    static constexpr int TP = PL::TP;
    static constexpr bool LAST = (S == PL::NP - 1);
    __device__ __forceinline__ static void run(cplx (&v)[E], cplx* sm0, cplx* sm1, int i, int team, const cplx* __restrict__ stw) {
#pragma unroll
        for (int m = 0; m < E / R; ++m) {
            const int b = i + TP * m;
            const int k = b & (P - 1);
            if constexpr (S > 0) {
                const cplx* __restrict__ t = stw + XCfg<N>::tw_offset(S) + k;
                if constexpr (R == 8 && MHD_XF_TWCHAIN == 3 && P >= 32) {
                    // w, w^2, w^4 from the table (3 reads), the other four powers by one multiplication each (depth 1)
                    cplx w1 = t[0], w2 = t[P], w4 = t[3 * P];
                    if (INV) { w1.y = -w1.y; w2.y = -w2.y; w4.y = -w4.y; }
                    const cplx w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4), w7 = cmul(w3, w4);
                    v[m * R + 1] = cmul(v[m * R + 1], w1); v[m * R + 2] = cmul(v[m * R + 2], w2);
                    v[m * R + 3] = cmul(v[m * R + 3], w3); v[m * R + 4] = cmul(v[m * R + 4], w4);
                    v[m * R + 5] = cmul(v[m * R + 5], w5); v[m * R + 6] = cmul(v[m * R + 6], w6);
                    v[m * R + 7] = cmul(v[m * R + 7], w7);
                } else if constexpr (R == 8 && (MHD_XF_TWCHAIN == 2 || (MHD_XF_TWCHAIN == 1 && P >= 32))) {
                    // the kernel is bound by shared-memory wavefronts, not FP64: read w and form w^2..w^7 by
                    // multiplication (depth <= 3, a few ulp) instead of 7 conflict-free but 4-wavefront reads
                    cplx w1 = t[0];
                    if (INV) w1.y = -w1.y;
                    const cplx w2 = cmul(w1, w1), w3 = cmul(w2, w1), w4 = cmul(w2, w2);
                    const cplx w5 = cmul(w4, w1), w6 = cmul(w3, w3), w7 = cmul(w4, w3);
                    v[m * R + 1] = cmul(v[m * R + 1], w1); v[m * R + 2] = cmul(v[m * R + 2], w2);
                    v[m * R + 3] = cmul(v[m * R + 3], w3); v[m * R + 4] = cmul(v[m * R + 4], w4);
                    v[m * R + 5] = cmul(v[m * R + 5], w5); v[m * R + 6] = cmul(v[m * R + 6], w6);
                    v[m * R + 7] = cmul(v[m * R + 7], w7);
                } else {
#pragma unroll
                    for (int q = 1; q < R; ++q) {
                        cplx w = t[(q - 1) * P];
                        if (INV) w.y = -w.y;
                        v[m * R + q] = cmul(v[m * R + q], w);
                    }
                }
            }
            bfly<R, INV>(&v[m * R]);
            if constexpr (!LAST) {
                if constexpr (P == 1) {            // first pass: j = R*b, element j + q
                    const int j = b * R, pj = xpad(j);
#pragma unroll
                    for (int q = 0; q < R; ++q) sm0[(R == 8) ? pj + q : xpad(j + q)] = v[m * R + q];
                } else {
                    const int j = (b - k) * R + k, pj = xpad(j);
#pragma unroll
                    for (int q = 0; q < R; ++q) sm0[(P % 8 == 0) ? pj + q * (P + P / 8) : xpad(j + q * P)] = v[m * R + q];
                }
            }
        }
        if constexpr (!LAST) {
            constexpr int Rn = PL::radix(S + 1);
            team_sync<TP>(team);
            const int pi = xpad(i);
#pragma unroll
            for (int m = 0; m < E / Rn; ++m)
#pragma unroll
                for (int q = 0; q < Rn; ++q) {
                    const int D = TP * m + q * (N / Rn);
                    v[m * Rn + q] = sm0[(D % 8 == 0) ? pi + D + D / 8 : xpad(i + D)];
                }
            if constexpr (SINGLE) team_sync<TP>(team);
            XPass<N, INV, S + 1, P * R, SINGLE>::run(v, sm1, sm0, i, team, stw);
        }
    }
};


// the thread's twiddles w of the radix-8 passes S >= 1 (8 points per thread: one butterfly per pass, k = i mod P): they do not
// depend on the row, so the x kernels read them from the shared tables once, before their row loop
template <int N> __device__ __forceinline__ void xpass2_own_twiddles(cplx (&wr)[4], int i, const cplx* __restrict__ stw) {
    using PL = Plan<N>;
    int P = PL::radix(0);
#pragma unroll
    for (int s = 1; s < 4; ++s) {
        wr[s] = make_double2(1.0, 0.0);
        if (s < PL::NP) {
            if (PL::radix(s) == 8) wr[s] = stw[XCfg<N>::tw_offset(s) + (i & (P - 1))];
            P *= PL::radix(s);
        }
    }
    wr[0] = make_double2(1.0, 0.0);
}

// Two independent transforms per thread (va, vb), pass by pass in lock step: the twiddles of a pass are formed once and
// applied to both, one team barrier serves both exchanges, and the two butterflies give every warp two independent
// instruction streams (the fused x pass is latency-bound: 12 warps per SM cannot cover the FP64 and shared-memory
// latencies of a single stream).  One exchange buffer per transform (smA, smB), two barriers per exchange.
template <int N, bool INV, int S, int P>
struct XPass2 {
    using PL = Plan<N>;
    static constexpr int R = PL::radix(S);
    static constexpr int E = PL::E;
    static constexpr int TP = PL::TP;
    static constexpr bool LAST = (S == PL::NP - 1);
    // wr[S]: the thread's own twiddle w of a radix-8 pass S (it depends on the slot i only), kept in registers by the caller
    __device__ __forceinline__ static void run(cplx (&va)[E], cplx (&vb)[E], cplx* smA, cplx* smB, int i, int team, const cplx* __restrict__ stw,
                                               const cplx (&wr)[4]) {
#pragma unroll
        for (int m = 0; m < E / R; ++m) {
            const int b = i + TP * m;
            const int k = b & (P - 1);
            if constexpr (S > 0) {
                const cplx* __restrict__ t = stw + XCfg<N>::tw_offset(S) + k;
                if constexpr (R == 8 && (MHD_XF2_TW == 2 || (MHD_XF2_TW == 3 && P >= 32) || (MHD_XF2_TW == 1 && P >= 32))) {
                    cplx w1 = (MHD_XF2_TWREG && E == 8) ? wr[S] : t[0], w2, w3, w4, w5, w6, w7;
                    if (INV) w1.y = -w1.y;
                    if constexpr (MHD_XF2_TW == 3) {      // w, w^2, w^4 from the table, four products of depth 1
                        w2 = t[P]; w4 = t[3 * P];
                        if (INV) { w2.y = -w2.y; w4.y = -w4.y; }
                        w3 = cmul(w1, w2); w5 = cmul(w1, w4); w6 = cmul(w2, w4); w7 = cmul(w3, w4);
                    } else {                              // everything from w (depth 3)
                        w2 = cmul(w1, w1); w3 = cmul(w2, w1); w4 = cmul(w2, w2);
                        w5 = cmul(w4, w1); w6 = cmul(w3, w3); w7 = cmul(w4, w3);
                    }
                    va[m * R + 1] = cmul(va[m * R + 1], w1); vb[m * R + 1] = cmul(vb[m * R + 1], w1);
                    va[m * R + 2] = cmul(va[m * R + 2], w2); vb[m * R + 2] = cmul(vb[m * R + 2], w2);
                    va[m * R + 3] = cmul(va[m * R + 3], w3); vb[m * R + 3] = cmul(vb[m * R + 3], w3);
                    va[m * R + 4] = cmul(va[m * R + 4], w4); vb[m * R + 4] = cmul(vb[m * R + 4], w4);
                    va[m * R + 5] = cmul(va[m * R + 5], w5); vb[m * R + 5] = cmul(vb[m * R + 5], w5);
                    va[m * R + 6] = cmul(va[m * R + 6], w6); vb[m * R + 6] = cmul(vb[m * R + 6], w6);
                    va[m * R + 7] = cmul(va[m * R + 7], w7); vb[m * R + 7] = cmul(vb[m * R + 7], w7);
                } else {
#pragma unroll
                    for (int q = 1; q < R; ++q) {
                        cplx w = t[(q - 1) * P];
                        if (INV) w.y = -w.y;
                        va[m * R + q] = cmul(va[m * R + q], w);
                        vb[m * R + q] = cmul(vb[m * R + q], w);
                    }
                }
            }
            bfly<R, INV>(&va[m * R]);
            if constexpr (MHD_XF2_LATEBAR == 2 && !LAST) continue;     // (the second butterfly and the writes follow below)
            bfly<R, INV>(&vb[m * R]);
            if constexpr (!LAST) {
                if constexpr (MHD_XF2_LATEBAR) { if (m == 0) team_sync<TP>(team); }     // every reader of the buffers is done
                if constexpr (P == 1) {            // first pass: j = R*b, element j + q
                    const int j = b * R, pj = xpad(j);
#pragma unroll
                    for (int q = 0; q < R; ++q) {
                        const int o = (R == 8) ? pj + q : xpad(j + q);
                        smA[o] = va[m * R + q]; smB[o] = vb[m * R + q];
                    }
                } else {
                    const int j = (b - k) * R + k, pj = xpad(j);
#pragma unroll
                    for (int q = 0; q < R; ++q) {
                        const int o = (P % 8 == 0) ? pj + q * (P + P / 8) : xpad(j + q * P);
                        smA[o] = va[m * R + q]; smB[o] = vb[m * R + q];
                    }
                }
            }
        }
        if constexpr (MHD_XF2_LATEBAR == 2 && !LAST) {
            // de-bursted order: A's writes are issued, then B's butterflies run while the load-store pipe drains them
            team_sync<TP>(team);
#pragma unroll
            for (int m = 0; m < E / R; ++m) {
                const int b = i + TP * m, k = b & (P - 1);
                const int j = (P == 1) ? b * R : (b - k) * R + k, pj = xpad(j);
#pragma unroll
                for (int q = 0; q < R; ++q) {
                    const int o = (P == 1) ? ((R == 8) ? pj + q : xpad(j + q)) : ((P % 8 == 0) ? pj + q * (P + P / 8) : xpad(j + q * P));
                    smA[o] = va[m * R + q];
                }
            }
#pragma unroll
            for (int e = 0; e < E; ++e) asm volatile("" : "+d"(vb[e].x), "+d"(vb[e].y));     // keep B's butterflies behind the barrier
#pragma unroll
            for (int m = 0; m < E / R; ++m) bfly<R, INV>(&vb[m * R]);
#pragma unroll
            for (int m = 0; m < E / R; ++m) {
                const int b = i + TP * m, k = b & (P - 1);
                const int j = (P == 1) ? b * R : (b - k) * R + k, pj = xpad(j);
#pragma unroll
                for (int q = 0; q < R; ++q) {
                    const int o = (P == 1) ? ((R == 8) ? pj + q : xpad(j + q)) : ((P % 8 == 0) ? pj + q * (P + P / 8) : xpad(j + q * P));
                    smB[o] = vb[m * R + q];
                }
            }
        }
        if constexpr (!LAST) {
            constexpr int Rn = PL::radix(S + 1);
            team_sync<TP>(team);
            const int pi = xpad(i);
#pragma unroll
            for (int m = 0; m < E / Rn; ++m)
#pragma unroll
                for (int q = 0; q < Rn; ++q) {
                    const int D = TP * m + q * (N / Rn);
                    const int o = (D % 8 == 0) ? pi + D + D / 8 : xpad(i + D);
                    va[m * Rn + q] = smA[o]; vb[m * Rn + q] = smB[o];
                }
            if constexpr (!MHD_XF2_LATEBAR) team_sync<TP>(team);
            XPass2<N, INV, S + 1, P * R>::run(va, vb, smA, smB, i, team, stw, wr);
        }
    }
};

}  // namespace mhd
