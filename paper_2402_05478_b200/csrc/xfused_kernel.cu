// xfused_kernel.cu — the fused x-pencil pass of the MHD step (SURVEY.md §8(a) S1-x + S2 + S3-x):
//
//     7 half-spectrum rows  --C2R-->  rho, m, B on N grid points  --products-->  12 real rows
//     --R2C-->  12 half-spectrum rows,     all inside one team of threads; real-space data never leaves registers.
//
// eq. (2) PAPER.md:41 (rho u u + (B^2/2) I - B B), eq. (4) PAPER.md:47 (u x B), u = m/rho for the
// viscous term; "products formed in real space" PAPER.md:78.
//
// Design (round-1 ncu of the first version: 255 registers, 8 warps/SM, 79 % of cycles without an
// eligible warp, a third of the stalls on the row loads; see profiles/r01_summary.md):
//   * persistent CTAs, one per SM, of TEAMS independent teams; a TEAM of TP = N/8 threads owns one
//     (z,y) row at a time (N = 512: 64 threads = 2 warps, 6 teams = 12 warps per SM).  Teams
//     synchronise among themselves only (named barrier, or __syncwarp when a team fits a warp), so the
//     FP64 phase of one team overlaps the shared-memory exchange of another.
//   * two real fields share one complex transform (Z = A + iB) both ways.  Every thread keeps 8
//     grid points x = i + TP*j of the 7 fields in registers: the inverse transform's last pass
//     leaves exactly the set the forward transform's first pass consumes, so the products are
//     thread-local.
//   * between passes the data is exchanged through two alternating team-private padded buffers, so one
//     barrier per exchange suffices; all shared-memory indices are a per-thread base plus
//     compile-time offsets.
//   * twiddles are read from per-pass shared tables laid out [leg][k] (conflict-free / broadcast).
//   * the Hermitian split after a forward transform needs Z[N-k] only: 3 of the 8 outputs go through
//     shared memory, Z[k] is already in the thread's own registers.
//   * the rows of the next field pairs (and of the team's next row) are pulled into L1 with
//     prefetch.global.L1 while the current transform runs, so the row loads hit L1.
// HBM traffic: reads 7 rows of nkx complex, writes 12 rows of nkx complex, in place in the same
// [field][row][px] array (a row's inputs are all consumed before its outputs are written).
#include "mhd_internal.h"
#include "xteam.cuh"

#ifndef MHD_XF_PREFETCH
#define MHD_XF_PREFETCH 1
#endif
// MHD_XF_THREADS (xteam.cuh): threads per persistent CTA for N >= 256 (a multiple of 128): 384 = 6 rows in flight per SM at N = 512
// MHD_XF_TWCHAIN (xteam.cuh): the kernel is bound by shared-memory wavefronts (80 % of the LSU data pipe), not FP64 (43 %): 2 is
// fastest (B200, 512^3).

namespace mhd {
using namespace mhdfft;

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// ---- TMA bulk copy (cp.async.bulk, global -> shared) completing on an mbarrier ----
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "XF_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra XF_DONE_%=;\n"
        "bra XF_WAIT_%=;\n"
        "XF_DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// PRUNED: nkx <= 3*TP (always true under the 2/3 rule), so the first-pass inputs q = 3, 4 are identically zero, the
// split only needs k = i + TP*t with t <= 2, and the rows are staged through shared memory by TMA.
template <int N, bool HYDRO, bool PRUNED>
__global__ void __launch_bounds__(XCfg<N>::THREADS, 1) xfused_kernel(XFusedArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    using CF = XCfg<N>;
    static_assert(PL::E == 8 && PL::radix(0) == 8, "fused x pass needs 8 points per thread and a radix-8 first pass");
    constexpr int TP = PL::TP, E = 8;
    constexpr int RL = PL::radix(PL::NP - 1);
    constexpr int NIN = HYDRO ? 2 : 4, NOUT = HYDRO ? 5 : 6;
    const int team = threadIdx.x / TP, i = threadIdx.x % TP;
    cplx* const smbase = reinterpret_cast<cplx*>(smraw);
    cplx* const stw = smbase + (size_t)2 * CF::BUF * CF::TEAMS;
    cplx* bufA = smbase + (size_t)team * 2 * CF::BUF;
    cplx* bufB = bufA + CF::BUF;
    const int nkx = a.nkx;
    // TMA staging (PRUNED only): per team 2 buffers x 2 rows x px complex, and one mbarrier per buffer
    cplx* const stage = stw + (CF::NTW > 0 ? CF::NTW : 1) + (size_t)team * 4 * a.px;
    unsigned long long* const mbar = reinterpret_cast<unsigned long long*>(stw + (CF::NTW > 0 ? CF::NTW : 1) + (size_t)CF::TEAMS * 4 * a.px) + 2 * team;
    if (PRUNED && i == 0) { mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); }
    if (PRUNED) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");

    // ---- per-pass twiddle tables [leg q-1][k], k < P:  w_N^(k q N/(P R)) ----
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

    const long long row_stride = (long long)gridDim.x * CF::TEAMS;
    const int pf_lines = (nkx * (int)sizeof(cplx) + 127) / 128;     // 128-byte lines per row (rows are 128-byte aligned)
    const unsigned row_bytes = (unsigned)nkx * (unsigned)sizeof(cplx);
    (void)pf_lines;

    // issue the TMA copies of field pair `pair` of row `r` into staging buffer (pair & 1): one thread per team
    auto stage_pair = [&](long long r, int pair) {
        const cplx* src = a.w2 + r * a.px + (long long)(2 * pair) * a.field_stride;
        cplx* dst = stage + (size_t)(pair & 1) * 2 * a.px;
        const bool two = pair < 3;
        mbar_expect_tx(&mbar[pair & 1], two ? 2 * row_bytes : row_bytes);
        bulk_g2s(dst, src, row_bytes, &mbar[pair & 1]);
        if (two) bulk_g2s(dst + a.px, src + a.field_stride, row_bytes, &mbar[pair & 1]);
    };
    unsigned phase = 0;          // bit b = parity the next wait on mbar[b] expects
    if (PRUNED) {
        const long long row0 = (long long)blockIdx.x * CF::TEAMS + team;
        if (i == 0 && row0 < a.nrows) { stage_pair(row0, 0); stage_pair(row0, 1); }
    }

    for (long long row = (long long)blockIdx.x * CF::TEAMS + team; row - team < a.nrows; row += row_stride) {
        // (every team of a CTA runs the same number of iterations; a team past the end works on zeros)
        const bool ok = row < a.nrows;
        cplx* __restrict__ base = a.w2 + (ok ? row : 0) * a.px;

#if MHD_XF_PREFETCH
        if (!PRUNED && ok)
            for (int f = 2; f < (HYDRO ? 4 : NFIELD); ++f)
                for (int l = i; l < pf_lines; l += TP) prefetch_l1(reinterpret_cast<const char*>(base + (long long)f * a.field_stride) + 128 * l);
#endif

        double inv[E], mx[E], my[E], mz[E], bx[E], by[E], bz[E];
#pragma unroll
        for (int j = 0; j < E; ++j) { inv[j] = 1.0; mx[j] = 0.0; my[j] = 0.0; mz[j] = 0.0; bx[j] = 0.0; by[j] = 0.0; bz[j] = 0.0; }

        // ---- inverse: field pairs (rho, mx) (my, mz) (Bx, By) (Bz, -) ----
#pragma unroll 1
        for (int pair = 0; pair < NIN; ++pair) {
            const bool hasB = pair < 3;
            cplx v[E];
            if constexpr (PRUNED) {
                const cplx* __restrict__ A = stage + (size_t)(pair & 1) * 2 * a.px;
                const cplx* __restrict__ B = A + a.px;
                if (ok) { mbar_wait(&mbar[pair & 1], (phase >> (pair & 1)) & 1u); phase ^= 1u << (pair & 1); }
#pragma unroll
                for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q; q = 3, 4 lie in the pruned band
                    if (q == 3 || q == 4) { v[q] = make_double2(0.0, 0.0); continue; }
                    const int k = i + TP * q;
                    const bool lo = (q < 3) && k < nkx, hi = (q > 4) && (N - k) < nkx;
                    const int idx = (q < 3) ? k : N - k;
                    cplx x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
                    if (ok && (lo || hi)) { x = A[idx]; if (hasB) y = B[idx]; }
                    if (k == 0) { x.y = 0.0; y.y = 0.0; }                               // self-conjugate mode: Im ignored
                    v[q] = (q < 3) ? make_double2(x.x - y.y, x.y + y.x) : make_double2(x.x + y.y, y.x - x.y);
                }
            } else {
                const cplx* __restrict__ A = base + (long long)(2 * pair) * a.field_stride;
                const cplx* __restrict__ B = hasB ? A + a.field_stride : A;
#pragma unroll
                for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q
                    const int k = i + TP * q;
                    const bool lo = k < nkx, hi = (N - k) < nkx;
                    const int idx = lo ? k : N - k;
                    cplx x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
                    if (ok && (lo || hi)) { x = A[idx]; if (hasB) y = B[idx]; }
                    if (k == 0 || 2 * k == N) { x.y = 0.0; y.y = 0.0; }                 // self-conjugate modes: Im ignored
                    // lo: A + iB;   hi (and not lo): conj(A) + i conj(B)
                    v[q] = lo ? make_double2(x.x - y.y, x.y + y.x) : make_double2(x.x + y.y, y.x - x.y);
                }
            }
            XPass<N, true, 0, 1>::run(v, bufA, bufB, i, team, stw);
            if (odd_exchanges<N>()) { cplx* t = bufA; bufA = bufB; bufB = t; }
            if constexpr (PRUNED) {
                // staging buffer (pair & 1) is free again: the team has passed a barrier since reading it (a one-thread
                // team needs none).  Refill it with pair + 2 of this row, or with the team's next row.
                if constexpr (PL::NP == 1 && TP > 1) team_sync<TP>(team);
                if (i == 0 && ok) {
                    if (pair + 2 < NIN) stage_pair(row, pair + 2);
                    else if (row + row_stride < a.nrows) stage_pair(row + row_stride, pair + 2 - NIN);
                }
            }
            const double s = a.scale;
            // last-pass outputs: register m*RL + q holds x = i + TP*m + q*(N/RL) = i + TP*(m + q*(E/RL))
            switch (pair) {
                case 0:
#pragma unroll
                    for (int m = 0; m < E / RL; ++m)
#pragma unroll
                        for (int q = 0; q < RL; ++q) { inv[m + q * (E / RL)] = v[m * RL + q].x * s; mx[m + q * (E / RL)] = v[m * RL + q].y * s; }
                    break;
                case 1:
#pragma unroll
                    for (int m = 0; m < E / RL; ++m)
#pragma unroll
                        for (int q = 0; q < RL; ++q) { my[m + q * (E / RL)] = v[m * RL + q].x * s; mz[m + q * (E / RL)] = v[m * RL + q].y * s; }
                    break;
                case 2:
#pragma unroll
                    for (int m = 0; m < E / RL; ++m)
#pragma unroll
                        for (int q = 0; q < RL; ++q) { bx[m + q * (E / RL)] = v[m * RL + q].x * s; by[m + q * (E / RL)] = v[m * RL + q].y * s; }
                    break;
                default:
#pragma unroll
                    for (int m = 0; m < E / RL; ++m)
#pragma unroll
                        for (int q = 0; q < RL; ++q) bz[m + q * (E / RL)] = v[m * RL + q].x * s;
                    break;
            }
        }
#pragma unroll
        for (int j = 0; j < E; ++j) inv[j] = ok ? 1.0 / inv[j] : 1.0;

        // ---- forward: product pairs (ux,uy) (uz,Txx) (Tyy,Tzz) (Txy,Txz) (Tyz,Ex) (Ey,Ez) ----
#pragma unroll 1
        for (int fp = 0; fp < NOUT; ++fp) {
            cplx v[E];
            int ida, idb;
            // keep the compiler from hoisting the (loop-invariant) products out of this rolled loop and spilling them
#pragma unroll
            for (int j = 0; j < E; ++j) {
                asm volatile("" : "+d"(inv[j]));
                if constexpr (!HYDRO) asm volatile("" : "+d"(bx[j]), "+d"(by[j]), "+d"(bz[j]));
            }
            switch (fp) {
                case 0:
                    ida = P_UX; idb = P_UY;
#pragma unroll
                    for (int j = 0; j < E; ++j) v[j] = make_double2(mx[j] * inv[j], my[j] * inv[j]);
                    break;
                case 1:
                    ida = P_UZ; idb = P_TXX;
#pragma unroll
                    for (int j = 0; j < E; ++j)
                        v[j] = make_double2(mz[j] * inv[j], mx[j] * (mx[j] * inv[j]) + 0.5 * (bx[j] * bx[j] + by[j] * by[j] + bz[j] * bz[j]) - bx[j] * bx[j]);
                    break;
                case 2:
                    ida = P_TYY; idb = P_TZZ;
#pragma unroll
                    for (int j = 0; j < E; ++j) {
                        const double b2h = 0.5 * (bx[j] * bx[j] + by[j] * by[j] + bz[j] * bz[j]);
                        v[j] = make_double2(my[j] * (my[j] * inv[j]) + b2h - by[j] * by[j], mz[j] * (mz[j] * inv[j]) + b2h - bz[j] * bz[j]);
                    }
                    break;
                case 3:
                    ida = P_TXY; idb = P_TXZ;
#pragma unroll
                    for (int j = 0; j < E; ++j) v[j] = make_double2(mx[j] * (my[j] * inv[j]) - bx[j] * by[j], mx[j] * (mz[j] * inv[j]) - bx[j] * bz[j]);
                    break;
                case 4:
                    ida = P_TYZ; idb = HYDRO ? -1 : P_EX;
#pragma unroll
                    for (int j = 0; j < E; ++j)
                        v[j] = make_double2(my[j] * (mz[j] * inv[j]) - by[j] * bz[j], HYDRO ? 0.0 : (my[j] * inv[j]) * bz[j] - (mz[j] * inv[j]) * by[j]);
                    break;
                default:
                    ida = P_EY; idb = P_EZ;
#pragma unroll
                    for (int j = 0; j < E; ++j)
                        v[j] = make_double2((mz[j] * inv[j]) * bx[j] - (mx[j] * inv[j]) * bz[j], (mx[j] * inv[j]) * by[j] - (my[j] * inv[j]) * bx[j]);
                    break;
            }
#if MHD_XF_PREFETCH
            if (!PRUNED && fp == NOUT - 2 && row + row_stride < a.nrows) {       // next row of this team: first two field pairs
                const cplx* nb = a.w2 + (row + row_stride) * a.px;
                for (int f = 0; f < (HYDRO ? 2 : 4); ++f)
                    for (int l = i; l < pf_lines; l += TP) prefetch_l1(reinterpret_cast<const char*>(nb + (long long)f * a.field_stride) + 128 * l);
            }
#endif
            // first-pass input register q must hold x = i + TP*q: that is how v was filled (j = q)
            XPass<N, false, 0, 1>::run(v, bufA, bufB, i, team, stw);
            if (odd_exchanges<N>()) { cplx* t = bufA; bufA = bufB; bufB = t; }
            // Hermitian split: A[k] = (Z[k] + conj Z[N-k])/2, B[k] = (Z[k] - conj Z[N-k])/(2i), k = i + TP*t < nkx.
            // Z[k] is this thread's own last-pass output; only Z[N-k] (held by slot (TP-i)%TP) crosses threads.
            // last-pass register m*RL + q holds index i + TP*(m + q*(E/RL)); publish those some k' = N-k can ask for.
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int t = m + q * (E / RL);            // index i + TP*t
                    if (PRUNED && t < 5) continue;                   // N - k > N - nkx >= 5*TP
                    if (t >= 1 && (TP * (t + 1) > N - nkx)) bufA[N - (i + TP * t)] = v[m * RL + q];   // index range [TP*t, TP*t+TP) meets [N-nkx+1, N)
                }
            team_sync<TP>(team);
            if (ok) {
                cplx* __restrict__ oa = base + (long long)ida * a.field_stride;
                cplx* __restrict__ ob = base + (long long)(idb < 0 ? 0 : idb) * a.field_stride;
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int t = m + q * (E / RL);
                        const int k = i + TP * t;
                        if (t <= (PRUNED ? 2 : E / 2) && k < nkx) {
                            const cplx zk = v[m * RL + q];
                            const cplx zm = (k == 0) ? zk : bufA[k];      // Z[N-k], published at position N - index (unpadded: conflict-free both ways)
                            oa[k] = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
                            if (idb >= 0) ob[k] = make_double2(0.5 * (zk.y + zm.y), 0.5 * (zm.x - zk.x));
                        }
                    }
            }
            { cplx* t = bufA; bufA = bufB; bufB = t; }
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
    cplx* bufA = smbase + (size_t)team * 2 * CF::BUF;
    cplx* bufB = bufA + CF::BUF;
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
            for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q
                const int k = i + TP * q;
                const bool lo = k < nkx, hi = (N - k) < nkx;
                const int idx = lo ? k : N - k;
                cplx x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
                if (ok && (lo || hi)) { x = A[idx]; y = B[idx]; }
                if (k == 0 || 2 * k == N) { x.y = 0.0; y.y = 0.0; }                 // self-conjugate modes: Im ignored
                v[q] = lo ? make_double2(x.x - y.y, x.y + y.x) : make_double2(x.x + y.y, y.x - x.y);
            }
            XPass<N, true, 0, 1>::run(v, bufA, bufB, i, team, stw);
            if (odd_exchanges<N>()) { cplx* t = bufA; bufA = bufB; bufB = t; }
            const double s = a.scale;
            if (ok) {
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int x = i + TP * (m + q * (E / RL));
                        ra[x] = v[m * RL + q].x * s;
                        rb[x] = v[m * RL + q].y * s;
                    }
            }
        } else {
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = ok ? make_double2(ra[i + TP * q], rb[i + TP * q]) : make_double2(0.0, 0.0);
            XPass<N, false, 0, 1>::run(v, bufA, bufB, i, team, stw);
            if (odd_exchanges<N>()) { cplx* t = bufA; bufA = bufB; bufB = t; }
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int t = m + q * (E / RL);
                    if (t >= 1 && (TP * (t + 1) > N - nkx)) bufA[N - (i + TP * t)] = v[m * RL + q];
                }
            team_sync<TP>(team);
            const double s = 0.5 * a.scale;
            if (ok) {
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int t = m + q * (E / RL);
                        const int k = i + TP * t;
                        if (t <= E / 2 && k < nkx) {
                            const cplx zk = v[m * RL + q];
                            const cplx zm = (k == 0) ? zk : bufA[k];
                            A[k] = make_double2(s * (zk.x + zm.x), s * (zk.y - zm.y));
                            B[k] = make_double2(s * (zk.y + zm.y), s * (zm.x - zk.x));
                        }
                    }
            }
            { cplx* t = bufA; bufA = bufB; bufB = t; }
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
        const long long groups = ((a.nrows + 1) / 2 + RC::TEAMS - 1) / RC::TEAMS;
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
        using CF = XCfg<N>;
        constexpr size_t kMaxSmem = 227 * 1024;
        // staged (TMA) rows need 2 buffers x 2 rows x px complex per team + the mbarriers
        const bool pruned = a.nkx <= 3 * CF::TP;
        const size_t smem = CF::SMEM + (pruned ? sizeof(cplx) * (size_t)CF::TEAMS * 4 * a.px + 16 * (size_t)CF::TEAMS : 0);
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
