// xfused_kernel.cu — the fused x-pencil pass of the MHD step (SURVEY.md §8(a) S1-x + S2 + S3-x):
//
//     7 half-spectrum rows  --C2R-->  rho, m, B on N grid points  --products-->  12 real rows
//     --R2C-->  12 half-spectrum rows,     all inside one team of threads; real-space data never leaves registers.
//
// eq. (2) PAPER.md:41 (rho u u + (B^2/2) I - B B), eq. (4) PAPER.md:47 (u x B), u = m/rho for the
// viscous term; "products formed in real space" PAPER.md:78.
//
// Design (history and measurements: DESIGN.md §6, profiles/r02_experiments.md):
//   * persistent CTAs, one per SM, of TEAMS independent teams; a TEAM of TP = N/8 threads owns one
//     (z,y) row at a time (N = 512: 64 threads = 2 warps, 4 teams = 8 warps per SM, up to 255 registers).
//     Teams synchronise among themselves only (named barrier, or __syncwarp when a team fits a warp).
//   * two real fields share one complex transform (Z = A + iB) both ways.  Every thread keeps 8
//     grid points x = i + TP*j of the 7 fields in registers: the inverse transform's last pass
//     leaves exactly the set the forward transform's first pass consumes, so the products are
//     thread-local.
//   * TWO transforms are in flight per thread (XPass2): (rho+i mx | my+i mz), (Bx+i By | Bz) inverse and three pairs of
//     product pairs forward.  Round 1 (12 warps/SM, one dependent stream each) was latency-bound: 53 % FP64 / 66 % LSU
//     utilisation, and neither pipe's instruction count moved the time.  Two independent streams per warp, one set of
//     twiddles and one barrier for both took it from 5.5 to 4.6 ms at 512^3 (LSU 72 % busy); four at once in the inverse
//     half gains nothing more (a round of four costs what two rounds of two do: throughput-bound now).
//   * between passes the data is exchanged through one team-private padded buffer per transform in flight; all
//     shared-memory indices are a per-thread base plus compile-time offsets.
//   * twiddles: w of a pass from a per-pass shared table laid out [leg][k], w^2..w^7 by multiplication.
//   * the Hermitian split after a forward transform needs Z[N-k] only: 3 of the 8 outputs go through
//     shared memory, Z[k] is already in the thread's own registers.
//   * the 7 input rows of a team's NEXT row are staged into shared memory by TMA (cp.async.bulk + mbarrier) while the
//     current row is transformed, one staging area per field group.
// HBM traffic: reads 7 rows of nkx complex, writes 12 rows of nkx complex, in place in the same
// [field][row][px] array (a row's inputs are all consumed before its outputs are written).
#include "mhd_internal.h"
#include "xteam.cuh"
#include "bulk_copy.cuh"

namespace mhd {
using namespace mhdfft;

// threads per persistent CTA of the fused pass for N >= 256: 256 = 4 rows in flight per SM at N = 512 (8 warps, up to 255 registers), each with two
// transforms in flight per thread (XPass2)
#ifndef MHD_XF2_THREADS
#define MHD_XF2_THREADS 256
#endif
template <int N> struct XCfg2 {
    static constexpr int TP = Plan<N>::TP;
    static constexpr int THREADS = (N >= 256) ? (MHD_XF2_THREADS / TP > 0 ? (MHD_XF2_THREADS / TP) * TP : TP) : 128;
    static constexpr int TEAMS = THREADS / TP;
    static constexpr int BUF = Padded::size(N);
    static constexpr int NTW = XCfg<N>::NTW > 0 ? XCfg<N>::NTW : 1;
    static constexpr size_t SMEM = sizeof(cplx) * ((size_t)2 * BUF * TEAMS + NTW);     // one exchange buffer per transform in flight
};

// PRUNED: nkx <= 3*TP (always true under the 2/3 rule), so the first-pass inputs q = 3, 4 are identically zero, the
// split only needs k = i + TP*t with t <= 2, and the rows are staged through shared memory by TMA: two staging areas per
// team, one per field group (rho, mx, my, mz | Bx, By, Bz), each refilled for the team's next row as soon as it is consumed.
template <int N, bool HYDRO, bool PRUNED>
__global__ void __launch_bounds__(XCfg2<N>::THREADS, 1) xfused_kernel(XFusedArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    using CF = XCfg2<N>;
    static_assert(PL::E == 8 && PL::radix(0) == 8, "fused x pass needs 8 points per thread and a radix-8 first pass");
    constexpr int TP = PL::TP, E = 8;
    constexpr int RL = PL::radix(PL::NP - 1);
    constexpr int NGRP = HYDRO ? 1 : 2;       // inverse: (rho,mx | my,mz) and (Bx,By | Bz,-)
    constexpr int NFWD = 3;                   // forward: (ux,uy | uz,Txx) (Tyy,Tzz | Txy,Txz) (Tyz,Ex | Ey,Ez); hydro: (Tyz,- | -,-)
    const int team = threadIdx.x / TP, i = threadIdx.x % TP;
    cplx* const smbase = reinterpret_cast<cplx*>(smraw);
    cplx* const stw = smbase + (size_t)2 * CF::BUF * CF::TEAMS;
    cplx* const bufA = smbase + (size_t)team * 2 * CF::BUF;
    cplx* const bufB = bufA + CF::BUF;
    const int nkx = a.nkx;
    // TMA staging (PRUNED only): per team 2 groups x 4 rows x px complex, and one mbarrier per group
    cplx* const stage = stw + CF::NTW + (size_t)team * 8 * a.px;
    unsigned long long* const mbar = reinterpret_cast<unsigned long long*>(stw + CF::NTW + (size_t)CF::TEAMS * 8 * a.px) + 2 * team;
    if (PRUNED && i == 0) { mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); }
    if (PRUNED) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");

    // ---- per-pass twiddle tables [leg q-1][k], k < P:  w_N^(k q N/(P R)) ----
    {
        int P = PL::radix(0);
#pragma unroll
        for (int s = 1; s < PL::NP; ++s) {
            const int R = PL::radix(s), off = XCfg<N>::tw_offset(s);
            for (int e = threadIdx.x; e < (R - 1) * P; e += blockDim.x) {
                const int q = e / P + 1, k = e % P;
                stw[off + e] = tw[k * q * (N / (P * R))];
            }
            P *= R;
        }
    }
    __syncthreads();
    cplx wr[4];
    xpass2_own_twiddles<N>(wr, i, stw);

    const long long row_stride = (long long)gridDim.x * CF::TEAMS;
    const unsigned row_bytes = (unsigned)nkx * (unsigned)sizeof(cplx);

    // issue the TMA copies of field group `grp` of row `r` into its staging area: one thread per team
    auto stage_group = [&](long long r, int grp) {
        const int nf = (grp == 0) ? 4 : 3;
        const cplx* src = a.w2 + r * a.px + (long long)(4 * grp) * a.field_stride;
        cplx* dst = stage + (size_t)grp * 4 * a.px;
        mbar_expect_tx(&mbar[grp], (unsigned)nf * row_bytes);
        for (int f = 0; f < nf; ++f) bulk_g2s(dst + (size_t)f * a.px, src + (long long)f * a.field_stride, row_bytes, &mbar[grp]);
    };
    unsigned phase = 0;          // bit g = parity the next wait on mbar[g] expects
    if (PRUNED) {
        const long long row0 = (long long)blockIdx.x * CF::TEAMS + team;
        if (i == 0 && row0 < a.nrows) { stage_group(row0, 0); if (!HYDRO) stage_group(row0, 1); }
    }

    for (long long row = (long long)blockIdx.x * CF::TEAMS + team; row - team < a.nrows; row += row_stride) {
        // (every team of a CTA runs the same number of iterations; a team past the end works on zeros)
        const bool ok = row < a.nrows;
        cplx* __restrict__ base = a.w2 + (ok ? row : 0) * a.px;

        double inv[E], mx[E], my[E], mz[E], bx[E], by[E], bz[E];
#pragma unroll
        for (int j = 0; j < E; ++j) { inv[j] = 1.0; mx[j] = 0.0; my[j] = 0.0; mz[j] = 0.0; bx[j] = 0.0; by[j] = 0.0; bz[j] = 0.0; }

        // ---- inverse: two transforms at a time, (rho + i mx | my + i mz) then (Bx + i By | Bz) ----
#pragma unroll
        for (int grp = 0; grp < NGRP; ++grp) {
            cplx va[E], vb[E];
            // rows of this group: A0 + i A1 -> va, B0 + i B1 -> vb (B1 absent in the magnetic group)
            const bool hasB1 = (grp == 0);
            if constexpr (PRUNED) {
                const cplx* __restrict__ S0 = stage + (size_t)grp * 4 * a.px;
                if (ok) { mbar_wait(&mbar[grp], (phase >> grp) & 1u); phase ^= 1u << grp; }
#pragma unroll
                for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q; q = 3, 4 lie in the pruned band
                    if (q == 3 || q == 4) { va[q] = make_double2(0.0, 0.0); vb[q] = make_double2(0.0, 0.0); continue; }
                    const int k = i + TP * q;
                    const bool lo = (q < 3) && k < nkx, hi = (q > 4) && (N - k) < nkx;
                    const int idx = (q < 3) ? k : N - k;
                    cplx x0 = make_double2(0.0, 0.0), x1 = x0, y0 = x0, y1 = x0;
                    if (ok && (lo || hi)) {
                        x0 = S0[idx]; x1 = S0[a.px + idx]; y0 = S0[2 * a.px + idx];
                        if (hasB1) y1 = S0[3 * a.px + idx];
                    }
                    if (k == 0) { x0.y = 0.0; x1.y = 0.0; y0.y = 0.0; y1.y = 0.0; }                       // self-conjugate mode: Im ignored
                    va[q] = (q < 3) ? make_double2(x0.x - x1.y, x0.y + x1.x) : make_double2(x0.x + x1.y, x1.x - x0.y);
                    vb[q] = (q < 3) ? make_double2(y0.x - y1.y, y0.y + y1.x) : make_double2(y0.x + y1.y, y1.x - y0.y);
                }
            } else {
                const cplx* __restrict__ G0 = base + (long long)(4 * grp) * a.field_stride;
#pragma unroll
                for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q
                    const int k = i + TP * q;
                    const bool lo = k < nkx, hi = (N - k) < nkx;
                    const int idx = lo ? k : N - k;
                    cplx x0 = make_double2(0.0, 0.0), x1 = x0, y0 = x0, y1 = x0;
                    if (ok && (lo || hi)) {
                        x0 = G0[idx]; x1 = G0[a.field_stride + idx]; y0 = G0[2 * a.field_stride + idx];
                        if (hasB1) y1 = G0[3 * a.field_stride + idx];
                    }
                    if (k == 0 || 2 * k == N) { x0.y = 0.0; x1.y = 0.0; y0.y = 0.0; y1.y = 0.0; }       // self-conjugate modes: Im ignored
                    // lo: A + iB;   hi (and not lo): conj(A) + i conj(B)
                    va[q] = lo ? make_double2(x0.x - x1.y, x0.y + x1.x) : make_double2(x0.x + x1.y, x1.x - x0.y);
                    vb[q] = lo ? make_double2(y0.x - y1.y, y0.y + y1.x) : make_double2(y0.x + y1.y, y1.x - y0.y);
                }
            }
            XPass2<N, true, 0, 1>::run(va, vb, bufA, bufB, i, team, stw, wr);
            if constexpr (PRUNED) {
                // the staging area of this group is free again: the team has passed a barrier since reading it (a one-thread
                // team needs none).  Refill it with the same group of the team's next row.
                if constexpr (PL::NP == 1 && TP > 1) team_sync<TP>(team);
                // (the team barrier orders the other threads' ld.shared before this point; the proxy fence orders those
                // generic-proxy reads before the async-proxy writes of the bulk copies issued next)
                if (i == 0 && ok && row + row_stride < a.nrows) { fence_proxy_async(); stage_group(row + row_stride, grp); }
            }
            const double s = a.scale;
            // last-pass outputs: register m*RL + q holds x = i + TP*m + q*(N/RL) = i + TP*(m + q*(E/RL))
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int j = m + q * (E / RL), r = m * RL + q;
                    if (grp == 0) { inv[j] = va[r].x * s; mx[j] = va[r].y * s; my[j] = vb[r].x * s; mz[j] = vb[r].y * s; }
                    else { bx[j] = va[r].x * s; by[j] = va[r].y * s; bz[j] = vb[r].x * s; }
                }
        }
#pragma unroll
        for (int j = 0; j < E; ++j) inv[j] = ok ? 1.0 / inv[j] : 1.0;

        // ---- forward: four products (two transforms) at a time ----
#pragma unroll 1
        for (int it = 0; it < NFWD; ++it) {
            cplx va[E], vb[E];
            int ida, idb, idc, idd;            // output fields of va.re, va.im, vb.re, vb.im (-1: none)
            // keep the compiler from hoisting the (loop-invariant) products out of this rolled loop and spilling them
#pragma unroll
            for (int j = 0; j < E; ++j) {
                asm volatile("" : "+d"(inv[j]));
                if constexpr (!HYDRO) asm volatile("" : "+d"(bx[j]), "+d"(by[j]), "+d"(bz[j]));
            }
            switch (it) {
                case 0:
                    ida = P_UX; idb = P_UY; idc = P_UZ; idd = P_TXX;
#pragma unroll
                    for (int j = 0; j < E; ++j) {
                        va[j] = make_double2(mx[j] * inv[j], my[j] * inv[j]);
                        vb[j] = make_double2(mz[j] * inv[j], mx[j] * (mx[j] * inv[j]) + 0.5 * (bx[j] * bx[j] + by[j] * by[j] + bz[j] * bz[j]) - bx[j] * bx[j]);
                    }
                    break;
                case 1:
                    ida = P_TYY; idb = P_TZZ; idc = P_TXY; idd = P_TXZ;
#pragma unroll
                    for (int j = 0; j < E; ++j) {
                        const double b2h = 0.5 * (bx[j] * bx[j] + by[j] * by[j] + bz[j] * bz[j]);
                        va[j] = make_double2(my[j] * (my[j] * inv[j]) + b2h - by[j] * by[j], mz[j] * (mz[j] * inv[j]) + b2h - bz[j] * bz[j]);
                        vb[j] = make_double2(mx[j] * (my[j] * inv[j]) - bx[j] * by[j], mx[j] * (mz[j] * inv[j]) - bx[j] * bz[j]);
                    }
                    break;
                default:
                    ida = P_TYZ; idb = HYDRO ? -1 : P_EX; idc = HYDRO ? -1 : P_EY; idd = HYDRO ? -1 : P_EZ;
#pragma unroll
                    for (int j = 0; j < E; ++j) {
                        va[j] = make_double2(my[j] * (mz[j] * inv[j]) - by[j] * bz[j], HYDRO ? 0.0 : (my[j] * inv[j]) * bz[j] - (mz[j] * inv[j]) * by[j]);
                        vb[j] = HYDRO ? make_double2(0.0, 0.0)
                                      : make_double2((mz[j] * inv[j]) * bx[j] - (mx[j] * inv[j]) * bz[j], (mx[j] * inv[j]) * by[j] - (my[j] * inv[j]) * bx[j]);
                    }
                    break;
            }
            // first-pass input register q must hold x = i + TP*q: that is how va, vb were filled (j = q)
            XPass2<N, false, 0, 1>::run(va, vb, bufA, bufB, i, team, stw, wr);
            // Hermitian split: A[k] = (Z[k] + conj Z[N-k])/2, B[k] = (Z[k] - conj Z[N-k])/(2i), k = i + TP*t < nkx.
            // Z[k] is this thread's own last-pass output; only Z[N-k] (held by slot (TP-i)%TP) crosses threads.
            // last-pass register m*RL + q holds index i + TP*(m + q*(E/RL)); publish those some k' = N-k can ask for.
            if constexpr (MHD_XF2_LATEBAR && PL::NP > 1) team_sync<TP>(team);     // the last exchange's reads are done
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int t = m + q * (E / RL);            // index i + TP*t
                    if (PRUNED && t < 5) continue;                   // N - k > N - nkx >= 5*TP
                    if (t >= 1 && (TP * (t + 1) > N - nkx)) {        // index range [TP*t, TP*t+TP) meets [N-nkx+1, N)
                        bufA[N - (i + TP * t)] = va[m * RL + q];
                        bufB[N - (i + TP * t)] = vb[m * RL + q];
                    }
                }
            team_sync<TP>(team);
            if (ok) {
                cplx* __restrict__ oa = base + (long long)ida * a.field_stride;
                cplx* __restrict__ ob = base + (long long)(idb < 0 ? 0 : idb) * a.field_stride;
                cplx* __restrict__ oc = base + (long long)(idc < 0 ? 0 : idc) * a.field_stride;
                cplx* __restrict__ od = base + (long long)(idd < 0 ? 0 : idd) * a.field_stride;
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int t = m + q * (E / RL);
                        const int k = i + TP * t;
                        if (t <= (PRUNED ? 2 : E / 2) && k < nkx) {
                            const cplx zk = va[m * RL + q];
                            const cplx zm = (k == 0) ? zk : bufA[k];      // Z[N-k], published at position N - index (unpadded: conflict-free both ways)
                            oa[k] = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
                            if (idb >= 0) ob[k] = make_double2(0.5 * (zk.y + zm.y), 0.5 * (zm.x - zk.x));
                            const cplx yk = vb[m * RL + q];
                            const cplx ym = (k == 0) ? yk : bufB[k];
                            if (idc >= 0) oc[k] = make_double2(0.5 * (yk.x + ym.x), 0.5 * (yk.y - ym.y));
                            if (idd >= 0) od[k] = make_double2(0.5 * (yk.y + ym.y), 0.5 * (ym.x - yk.x));
                        }
                    }
            }
            // the split reads are done before the next transform's first exchange writes the buffers (late-barrier passes
            // synchronise in front of every write themselves)
            if constexpr (!(MHD_XF2_LATEBAR && PL::NP > 1)) team_sync<TP>(team);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Stand-alone x pass on the same team machinery: pairs of real rows <-> pairs of half-spectrum rows (mhd_fft_r2c /
// mhd_fft_c2r of BASELINE config 5, mhd_set_fields, mhd_get_fields, diagnostics).  One team per row pair; consecutive
// lanes touch consecutive x (or kx), so every global access is a full line.  Little per-thread state => 256-thread CTAs,
// several per SM; persistent so the twiddle tables are built once per CTA.
template <int N> struct XRowCfg {
    static constexpr int TP = Plan<N>::TP;
    static constexpr int THREADS = (TP >= 128) ? 256 : 128 < TP ? TP : (N >= 256 ? 256 : 128);
    static constexpr int TEAMS = THREADS / TP;
    static constexpr size_t SMEM = sizeof(cplx) * ((size_t)2 * XCfg<N>::BUF * TEAMS + (XCfg<N>::NTW > 0 ? XCfg<N>::NTW : 1));
};

template <int N, bool INV>
__global__ void __launch_bounds__(XRowCfg<N>::THREADS) xrows_kernel(RowArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    using CF = XCfg<N>;
    using RC = XRowCfg<N>;
    constexpr int TP = PL::TP, E = 8;
    constexpr int RL = PL::radix(PL::NP - 1);
    const int team = threadIdx.x / TP, i = threadIdx.x % TP;
    cplx* const smbase = reinterpret_cast<cplx*>(smraw);
    cplx* const stw = smbase + (size_t)2 * CF::BUF * RC::TEAMS;
    cplx* const bufA = smbase + (size_t)team * 2 * CF::BUF;
    cplx* const bufB = bufA + CF::BUF;
    const int nkx = a.nkx;
    {
        int P = PL::radix(0);
#pragma unroll
        for (int s = 1; s < PL::NP; ++s) {
            const int R = PL::radix(s), off = CF::tw_offset(s);
            for (int e = threadIdx.x; e < (R - 1) * P; e += blockDim.x) {
                const int q = e / P + 1, k = e % P;
                stw[off + e] = tw[k * q * (N / (P * R))];
            }
            P *= R;
        }
    }
    __syncthreads();
    cplx wr[4];
    xpass2_own_twiddles<N>(wr, i, stw);
    // a team takes TWO row pairs per iteration (two transforms in flight per thread, XPass2): the kernel is latency-bound
    const long long npairs = (a.nrows + 1) / 2;
    const long long nunits = (npairs + 1) / 2;
    const long long stride = (long long)gridDim.x * RC::TEAMS;
    for (long long u = (long long)blockIdx.x * RC::TEAMS + team; u - team < nunits; u += stride) {
        const bool oka = 2 * u < npairs, okb = 2 * u + 1 < npairs;
        const long long r0 = oka ? 4 * u : 0, r1 = okb ? 4 * u + 2 : 0;
        cplx* __restrict__ A0 = a.spec + r0 * a.spec_pitch;
        cplx* __restrict__ A1 = A0 + a.spec_pitch;
        cplx* __restrict__ B0 = a.spec + r1 * a.spec_pitch;
        cplx* __restrict__ B1 = B0 + a.spec_pitch;
        double* __restrict__ ra0 = a.real + r0 * a.real_pitch;
        double* __restrict__ ra1 = ra0 + a.real_pitch;
        double* __restrict__ rb0 = a.real + r1 * a.real_pitch;
        double* __restrict__ rb1 = rb0 + a.real_pitch;
        cplx va[E], vb[E];
        if constexpr (INV) {
            // pull the team's NEXT four spectrum rows towards L2 while this unit is transformed: the inverse kernel's dominant stall
            // is the wait for these loads (ncu: long scoreboard).  Measured at 512^3 x 7: C2R 9.1 -> 8.9 ms; the same prefetch in
            // the forward direction costs 4 % (8.25 -> 8.55 ms) and is therefore not done.
            const long long un = u + stride;
            if (2 * un < npairs) {
                const char* nsrc = reinterpret_cast<const char*>(a.spec + 4 * un * a.spec_pitch);
                const long long left = a.nrows - 4 * un;                                   // rows that exist from there on
                const long long bytes = (left < 4 ? left : 4) * a.spec_pitch * (long long)sizeof(cplx);
                for (long long o = (long long)i * 128; o < bytes; o += (long long)TP * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(nsrc + o));
            }
        }
        if constexpr (INV) {
#pragma unroll
            for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q
                const int k = i + TP * q;
                const bool lo = k < nkx, hi = (N - k) < nkx;
                const int idx = lo ? k : N - k;
                cplx x0 = make_double2(0.0, 0.0), x1 = x0, y0 = x0, y1 = x0;
                if (lo || hi) {
                    if (oka) { x0 = A0[idx]; x1 = A1[idx]; }
                    if (okb) { y0 = B0[idx]; y1 = B1[idx]; }
                }
                if (k == 0 || 2 * k == N) { x0.y = 0.0; x1.y = 0.0; y0.y = 0.0; y1.y = 0.0; }   // self-conjugate modes: Im ignored
                va[q] = lo ? make_double2(x0.x - x1.y, x0.y + x1.x) : make_double2(x0.x + x1.y, x1.x - x0.y);
                vb[q] = lo ? make_double2(y0.x - y1.y, y0.y + y1.x) : make_double2(y0.x + y1.y, y1.x - y0.y);
            }
            XPass2<N, true, 0, 1>::run(va, vb, bufA, bufB, i, team, stw, wr);
            const double s = a.scale;
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int x = i + TP * (m + q * (E / RL));
                    if (oka) { ra0[x] = va[m * RL + q].x * s; ra1[x] = va[m * RL + q].y * s; }
                    if (okb) { rb0[x] = vb[m * RL + q].x * s; rb1[x] = vb[m * RL + q].y * s; }
                }
        } else {
#pragma unroll
            for (int q = 0; q < E; ++q) {
                va[q] = oka ? make_double2(ra0[i + TP * q], ra1[i + TP * q]) : make_double2(0.0, 0.0);
                vb[q] = okb ? make_double2(rb0[i + TP * q], rb1[i + TP * q]) : make_double2(0.0, 0.0);
            }
            XPass2<N, false, 0, 1>::run(va, vb, bufA, bufB, i, team, stw, wr);
            // Hermitian split: only Z[N-k] crosses threads (see the fused kernel)
            if constexpr (MHD_XF2_LATEBAR && PL::NP > 1) team_sync<TP>(team);
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int t = m + q * (E / RL);
                    if (t >= 1 && (TP * (t + 1) > N - nkx)) { bufA[N - (i + TP * t)] = va[m * RL + q]; bufB[N - (i + TP * t)] = vb[m * RL + q]; }
                }
            team_sync<TP>(team);
            const double s = 0.5 * a.scale;
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int t = m + q * (E / RL);
                    const int k = i + TP * t;
                    if (t <= E / 2 && k < nkx) {
                        if (oka) {
                            const cplx zk = va[m * RL + q];
                            const cplx zm = (k == 0) ? zk : bufA[k];
                            A0[k] = make_double2(s * (zk.x + zm.x), s * (zk.y - zm.y));
                            A1[k] = make_double2(s * (zk.y + zm.y), s * (zm.x - zk.x));
                        }
                        if (okb) {
                            const cplx zk = vb[m * RL + q];
                            const cplx zm = (k == 0) ? zk : bufB[k];
                            B0[k] = make_double2(s * (zk.x + zm.x), s * (zk.y - zm.y));
                            B1[k] = make_double2(s * (zk.y + zm.y), s * (zm.x - zk.x));
                        }
                    }
                }
            if constexpr (!(MHD_XF2_LATEBAR && PL::NP > 1)) team_sync<TP>(team);
        }
    }
}

// Inverse x rows with TMA-staged inputs (N >= 128, 8 points per thread): the plain inverse kernel above spends its time waiting
// for its row loads (ncu: long scoreboard, 56 % of the DRAM rate against 78 % for the forward direction).  Here one persistent
// CTA per SM runs the fused pass's scheme: a team's NEXT unit (four consecutive half-spectrum rows = one contiguous block) is
// brought into shared memory by one bulk copy (cp.async.bulk + mbarrier, two staging buffers per team) while the current unit
// is transformed, so no warp ever waits on a global load.
#ifndef MHD_XROWS_INV_STAGED
#define MHD_XROWS_INV_STAGED 1
#endif
#ifndef MHD_XROWS_INV_STAGED_MIN
#define MHD_XROWS_INV_STAGED_MIN 128     // shortest row length that takes the staged kernel
#endif
template <int N> struct XRowStagedCfg {
    static constexpr int TP = Plan<N>::TP;
    static constexpr int THREADS = 256;
    static constexpr int TEAMS = THREADS / TP;
    static constexpr int NTW = XCfg<N>::NTW > 0 ? XCfg<N>::NTW : 1;
    __host__ __device__ static size_t smem(long long pitch) {       // exchange buffers, twiddle tables, 2 x 4 staged rows per team, mbarriers
        return sizeof(cplx) * ((size_t)2 * XCfg<N>::BUF * TEAMS + NTW + (size_t)TEAMS * 8 * pitch) + 16 * (size_t)TEAMS;
    }
};

template <int N>
__global__ void __launch_bounds__(XRowStagedCfg<N>::THREADS, 1) xrows_inv_staged_kernel(RowArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    using CF = XCfg<N>;
    using RC = XRowStagedCfg<N>;
    static_assert(PL::E == 8 && RC::TEAMS >= 1, "staged inverse x rows: 8 points per thread");
    constexpr int TP = PL::TP, E = 8;
    constexpr int RL = PL::radix(PL::NP - 1);
    const int team = threadIdx.x / TP, i = threadIdx.x % TP;
    cplx* const smbase = reinterpret_cast<cplx*>(smraw);
    cplx* const stw = smbase + (size_t)2 * CF::BUF * RC::TEAMS;
    cplx* const bufA = smbase + (size_t)team * 2 * CF::BUF;
    cplx* const bufB = bufA + CF::BUF;
    const int nkx = a.nkx;
    const long long pitch = a.spec_pitch;
    cplx* const stage = stw + RC::NTW + (size_t)team * 8 * pitch;                  // two buffers of 4 rows
    unsigned long long* const mbar = reinterpret_cast<unsigned long long*>(stw + RC::NTW + (size_t)RC::TEAMS * 8 * pitch) + 2 * team;
    if (i == 0) { mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    {
        int P = PL::radix(0);
#pragma unroll
        for (int s = 1; s < PL::NP; ++s) {
            const int R = PL::radix(s), off = CF::tw_offset(s);
            for (int e = threadIdx.x; e < (R - 1) * P; e += blockDim.x) {
                const int q = e / P + 1, k = e % P;
                stw[off + e] = tw[k * q * (N / (P * R))];
            }
            P *= R;
        }
    }
    __syncthreads();
    cplx wr[4];
    xpass2_own_twiddles<N>(wr, i, stw);

    const long long npairs = (a.nrows + 1) / 2;
    const long long nunits = (npairs + 1) / 2;
    const long long stride = (long long)gridDim.x * RC::TEAMS;
    // rows 4u .. 4u+3 of unit u are one contiguous block of the spectrum array (fewer at the end of the batch)
    auto stage_unit = [&](long long u, int b) {
        const long long left = a.nrows - 4 * u;
        const unsigned bytes = (unsigned)((left < 4 ? left : 4) * pitch * (long long)sizeof(cplx));
        mbar_expect_tx(&mbar[b], bytes);
        bulk_g2s(stage + (size_t)b * 4 * pitch, a.spec + 4 * u * pitch, bytes, &mbar[b]);
    };
    const long long u0 = (long long)blockIdx.x * RC::TEAMS + team;
    if (i == 0 && u0 < nunits) stage_unit(u0, 0);
    unsigned phase = 0;          // bit b = parity the next wait on mbar[b] expects
    int b = 0;
    for (long long u = u0; u - team < nunits; u += stride, b ^= 1) {
        const bool oku = u < nunits;
        const bool oka = oku && 2 * u < npairs, okb = oku && 2 * u + 1 < npairs;
        // every thread of the team has finished reading buffer b^1 (it passed the team barriers of the previous transform)
        // (generic-proxy reads, then async-proxy writes of the same bytes: proxy fence in the issuing thread)
        if (i == 0 && u + stride < nunits) { fence_proxy_async(); stage_unit(u + stride, b ^ 1); }
        if (oku) { mbar_wait(&mbar[b], (phase >> b) & 1u); phase ^= 1u << b; }
        const cplx* __restrict__ A0 = stage + (size_t)b * 4 * pitch;
        const cplx* __restrict__ A1 = A0 + pitch;
        const cplx* __restrict__ B0 = A1 + pitch;
        const cplx* __restrict__ B1 = B0 + pitch;
        const long long r0 = oka ? 4 * u : 0, r1 = okb ? 4 * u + 2 : 0;
        double* __restrict__ ra0 = a.real + r0 * a.real_pitch;
        double* __restrict__ ra1 = ra0 + a.real_pitch;
        double* __restrict__ rb0 = a.real + r1 * a.real_pitch;
        double* __restrict__ rb1 = rb0 + a.real_pitch;
        cplx va[E], vb[E];
#pragma unroll
        for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q
            const int k = i + TP * q;
            const bool lo = k < nkx, hi = (N - k) < nkx;
            const int idx = lo ? k : N - k;
            cplx x0 = make_double2(0.0, 0.0), x1 = x0, y0 = x0, y1 = x0;
            if (lo || hi) {
                if (oka) { x0 = A0[idx]; x1 = A1[idx]; }
                if (okb) { y0 = B0[idx]; y1 = B1[idx]; }
            }
            if (k == 0 || 2 * k == N) { x0.y = 0.0; x1.y = 0.0; y0.y = 0.0; y1.y = 0.0; }   // self-conjugate modes: Im ignored
            va[q] = lo ? make_double2(x0.x - x1.y, x0.y + x1.x) : make_double2(x0.x + x1.y, x1.x - x0.y);
            vb[q] = lo ? make_double2(y0.x - y1.y, y0.y + y1.x) : make_double2(y0.x + y1.y, y1.x - y0.y);
        }
        XPass2<N, true, 0, 1>::run(va, vb, bufA, bufB, i, team, stw, wr);
        const double s = a.scale;
#pragma unroll
        for (int m = 0; m < E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int x = i + TP * (m + q * (E / RL));
                if (oka) { ra0[x] = va[m * RL + q].x * s; ra1[x] = va[m * RL + q].y * s; }
                if (okb) { rb0[x] = vb[m * RL + q].x * s; rb1[x] = vb[m * RL + q].y * s; }
            }
    }
}

// Lengths 3*2^a (12 or 24 points per thread, a radix-3 last pass): the same team machinery with one exchange buffer per
// team and general first/last-pass index sets.  128 threads per CTA (4 teams at N = 768), persistent.
template <int N> struct XRowGenCfg {
    static constexpr int TP = Plan<N>::TP;
    static constexpr int THREADS = 128;
    static constexpr int TEAMS = THREADS / TP;
    static constexpr size_t SMEM = sizeof(cplx) * ((size_t)XCfg<N>::BUF * TEAMS + (XCfg<N>::NTW > 0 ? XCfg<N>::NTW : 1));
};

template <int N, bool INV>
__global__ void __launch_bounds__(XRowGenCfg<N>::THREADS, 3) xrows_general_kernel(RowArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    using CF = XCfg<N>;
    using RC = XRowGenCfg<N>;
    constexpr int TP = PL::TP, E = PL::E;
    constexpr int R0 = PL::radix(0), RL = PL::radix(PL::NP - 1);
    const int team = threadIdx.x / TP, i = threadIdx.x % TP;
    cplx* const smbase = reinterpret_cast<cplx*>(smraw);
    cplx* const stw = smbase + (size_t)CF::BUF * RC::TEAMS;
    cplx* const buf = smbase + (size_t)team * CF::BUF;
    const int nkx = a.nkx;
    {
        int P = PL::radix(0);
#pragma unroll
        for (int s = 1; s < PL::NP; ++s) {
            const int R = PL::radix(s), off = CF::tw_offset(s);
            for (int e = threadIdx.x; e < (R - 1) * P; e += blockDim.x) {
                const int q = e / P + 1, k = e % P;
                stw[off + e] = tw[k * q * (N / (P * R))];
            }
            P *= R;
        }
    }
    __syncthreads();
    const long long npairs = (a.nrows + 1) / 2;
    const long long stride = (long long)gridDim.x * RC::TEAMS;
    for (long long pr = (long long)blockIdx.x * RC::TEAMS + team; pr - team < npairs; pr += stride) {
        const bool ok = pr < npairs;
        const long long r0 = ok ? 2 * pr : 0;
        cplx* __restrict__ A = a.spec + r0 * a.spec_pitch;
        cplx* __restrict__ B = A + a.spec_pitch;
        double* __restrict__ ra = a.real + r0 * a.real_pitch;
        double* __restrict__ rb = ra + a.real_pitch;
        cplx v[E];
        if constexpr (INV) {
#pragma unroll
            for (int m = 0; m < E / R0; ++m)
#pragma unroll
                for (int q = 0; q < R0; ++q) {
                    const int k = first_index<N>(i, m, q);
                    const bool lo = k < nkx, hi = (N - k) < nkx;
                    const int idx = lo ? k : N - k;
                    cplx x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
                    if (ok && (lo || hi)) { x = A[idx]; y = B[idx]; }
                    if (k == 0 || 2 * k == N) { x.y = 0.0; y.y = 0.0; }                 // self-conjugate modes: Im ignored
                    v[first_reg<N>(m, q)] = lo ? make_double2(x.x - y.y, x.y + y.x) : make_double2(x.x + y.y, y.x - x.y);
                }
            XPass<N, true, 0, 1, true>::run(v, buf, buf, i, team, stw);
            const double s = a.scale;
            if (ok) {
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int x = last_index<N>(i, m, q);
                        ra[x] = v[last_reg<N>(m, q)].x * s;
                        rb[x] = v[last_reg<N>(m, q)].y * s;
                    }
            }
        } else {
#pragma unroll
            for (int m = 0; m < E / R0; ++m)
#pragma unroll
                for (int q = 0; q < R0; ++q) {
                    const int x = first_index<N>(i, m, q);
                    v[first_reg<N>(m, q)] = ok ? make_double2(ra[x], rb[x]) : make_double2(0.0, 0.0);
                }
            XPass<N, false, 0, 1, true>::run(v, buf, buf, i, team, stw);
            // Hermitian split: publish Z[j] for the j some k = N - j < nkx will ask for, at position N - j (unpadded)
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int j = last_index<N>(i, m, q);
                    if (j >= 1 && N - j < nkx) buf[N - j] = v[last_reg<N>(m, q)];
                }
            team_sync<TP>(team);
            const double s = 0.5 * a.scale;
            if (ok) {
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int k = last_index<N>(i, m, q);
                        if (k < nkx && 2 * k <= N) {
                            const cplx zk = v[last_reg<N>(m, q)];
                            const cplx zm = (k == 0) ? zk : buf[k];
                            A[k] = make_double2(s * (zk.x + zm.x), s * (zk.y - zm.y));
                            B[k] = make_double2(s * (zk.y + zm.y), s * (zm.x - zk.x));
                        }
                    }
            }
            team_sync<TP>(team);
        }
    }
}

template <int N> static cudaError_t launch_xrows_n(bool inverse, const RowArgs& a, const cplx* tw, cudaStream_t st) {
    static DeviceOnce once;
    const int dev = device_slot();
    if (dev < 0) return cudaErrorInvalidDevice;
    int sms = 0;
    cudaError_t e = device_sm_count(dev, &sms);
    if (e != cudaSuccess) return e;
    if constexpr (Plan<N>::E != 8) {
        using RC = XRowGenCfg<N>;
        if (!once.done[dev]) {
            e = cudaFuncSetAttribute(xrows_general_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RC::SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(xrows_general_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RC::SMEM);
            if (e != cudaSuccess) return e;
            once.done[dev] = true;
        }
        const long long groups = ((a.nrows + 1) / 2 + RC::TEAMS - 1) / RC::TEAMS;
        const long long cap = (long long)sms * 8;
        const unsigned blocks = (unsigned)(groups < cap ? groups : cap);
        if (inverse) xrows_general_kernel<N, true><<<blocks, RC::THREADS, RC::SMEM, st>>>(a, tw);
        else xrows_general_kernel<N, false><<<blocks, RC::THREADS, RC::SMEM, st>>>(a, tw);
        count_launch();
        return cudaGetLastError();
    } else {
        using RC = XRowCfg<N>;
        if (!once.done[dev]) {
            e = cudaFuncSetAttribute(xrows_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RC::SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(xrows_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RC::SMEM);
            if (e != cudaSuccess) return e;
            once.done[dev] = true;
        }
        if constexpr (MHD_XROWS_INV_STAGED && N >= MHD_XROWS_INV_STAGED_MIN) {
            using SC = XRowStagedCfg<N>;
            const size_t smem = SC::smem(a.spec_pitch);
            // (bulk copies want 16-byte aligned rows: any complex pitch is; the array itself comes from a 256-byte aligned workspace)
            if (inverse && smem <= (size_t)227 * 1024 && a.nrows % 2 == 0 && ((size_t)a.spec & 15u) == 0) {
                static DeviceOnce once_staged;
                if (!once_staged.done[dev]) {
                    e = cudaFuncSetAttribute(xrows_inv_staged_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
                    if (e != cudaSuccess) return e;
                    once_staged.done[dev] = true;
                }
                const long long units = (((a.nrows + 1) / 2 + 1) / 2 + SC::TEAMS - 1) / SC::TEAMS;
                const unsigned nb = (unsigned)(units < sms ? units : sms);         // one persistent CTA per SM
                xrows_inv_staged_kernel<N><<<nb, SC::THREADS, smem, st>>>(a, tw);
                count_launch();
                return cudaGetLastError();
            }
        }
        const long long groups = (((a.nrows + 1) / 2 + 1) / 2 + RC::TEAMS - 1) / RC::TEAMS;   // two row pairs per team iteration
        const long long cap = (long long)sms * 8;             // persistent; more CTAs than can be resident simply queue
        const unsigned blocks = (unsigned)(groups < cap ? groups : cap);
        if (inverse) xrows_kernel<N, true><<<blocks, RC::THREADS, RC::SMEM, st>>>(a, tw);
        else xrows_kernel<N, false><<<blocks, RC::THREADS, RC::SMEM, st>>>(a, tw);
        count_launch();
        return cudaGetLastError();
    }
}

cudaError_t launch_xrows(int n, bool inverse, const RowArgs& a, const double2* tw, cudaStream_t st) {
    switch (n) {
#define X(N_) case N_: return launch_xrows_n<N_>(inverse, a, tw, st);
        X(8) X(12) X(16) X(24) X(32) X(48) X(64) X(96) X(128) X(192) X(256) X(384) X(512) X(768) X(1024)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

template <int N> static cudaError_t launch_xfused_n(const XFusedArgs& a, int hydro, const cplx* tw, cudaStream_t st) {
    if constexpr (Plan<N>::E != 8) {
        return cudaErrorInvalidValue;
    } else {
        using CF = XCfg2<N>;
        constexpr size_t kMaxSmem = 227 * 1024;
        // staged (TMA) rows need 2 groups x 4 rows x px complex per team + the mbarriers
        const bool pruned = a.nkx <= 3 * CF::TP;
        const size_t smem = CF::SMEM + (pruned ? sizeof(cplx) * (size_t)CF::TEAMS * 8 * a.px + 16 * (size_t)CF::TEAMS : 0);
        if (smem > kMaxSmem) return cudaErrorInvalidValue;
        static DeviceOnce once;
        const int dev = device_slot();
        if (dev < 0) return cudaErrorInvalidDevice;
        int sms = 0;
        cudaError_t e = device_sm_count(dev, &sms);
        if (e != cudaSuccess) return e;
        if (!once.done[dev]) {
            e = cudaFuncSetAttribute(xfused_kernel<N, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(xfused_kernel<N, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(xfused_kernel<N, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(xfused_kernel<N, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
            if (e != cudaSuccess) return e;
            once.done[dev] = true;
        }
        // persistent: one CTA per SM, or fewer when there are not enough rows; several CTAs per SM for the small lengths
        const long long groups = (a.nrows + CF::TEAMS - 1) / CF::TEAMS;
        const long long cap = (long long)sms * (N >= 256 ? 1 : 4);
        const unsigned blocks = (unsigned)(groups < cap ? groups : cap);
        if (pruned) {
            if (hydro) xfused_kernel<N, true, true><<<blocks, CF::THREADS, smem, st>>>(a, tw);
            else xfused_kernel<N, false, true><<<blocks, CF::THREADS, smem, st>>>(a, tw);
        } else {
            if (hydro) xfused_kernel<N, true, false><<<blocks, CF::THREADS, smem, st>>>(a, tw);
            else xfused_kernel<N, false, false><<<blocks, CF::THREADS, smem, st>>>(a, tw);
        }
        count_launch();
        return cudaGetLastError();
    }
}

bool xfused_supported(int n) {
    switch (n) {
        case 8: case 16: case 32: case 64: case 128: case 256: case 512: case 1024: return true;
        default: return false;
    }
}

cudaError_t launch_xfused(int n, const XFusedArgs& a, int hydro, const double2* tw, cudaStream_t st) {
    switch (n) {
        case 8: return launch_xfused_n<8>(a, hydro, tw, st);
        case 16: return launch_xfused_n<16>(a, hydro, tw, st);
        case 32: return launch_xfused_n<32>(a, hydro, tw, st);
        case 64: return launch_xfused_n<64>(a, hydro, tw, st);
        case 128: return launch_xfused_n<128>(a, hydro, tw, st);
        case 256: return launch_xfused_n<256>(a, hydro, tw, st);
        case 512: return launch_xfused_n<512>(a, hydro, tw, st);
        case 1024: return launch_xfused_n<1024>(a, hydro, tw, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace mhd
