// xfused_kernel.cu — the fused x-pencil pass of the MHD step (SURVEY.md §8(a) S1-x + S2 + S3-x):
//
//     7 half-spectrum rows  --C2R-->  rho, m, B on 512 grid points  --products-->  12 real rows
//     --R2C-->  12 half-spectrum rows,          all inside one CTA, real-space data never leaves registers.
//
// eq. (2) PAPER.md:41 (rho u u + (B^2/2) I - B B), eq. (4) PAPER.md:47 (u x B), u = m/rho for the
// viscous term; "products formed in real space" PAPER.md:78.
//
// One TEAM of TP = N/8 threads owns one (z,y) row (N = 512: 64 threads = 2 warps = one CTA).  Two
// real fields share one complex transform (Z = A + iB).  Every thread keeps 8 grid points of each
// of the 7 fields: the inverse transform leaves slot i with x = i + TP*j, j = 0..7, and the forward
// transform wants exactly the same set as its first-pass input, so the products are thread-local.
// Each transform exchanges data between passes through a team-private padded shared buffer.
// HBM traffic: reads 7 rows of nkx complex, writes 12 rows of nkx complex, in place in the same
// [field][row][px] array (a row's inputs are all consumed before its outputs are written).
#include "mhd_internal.h"
#include "fft_core.cuh"

// resident CTAs per SM the register allocator is asked to allow (tuning knob)
#ifndef MHD_XFUSED_MINBLOCKS
#define MHD_XFUSED_MINBLOCKS 1
#endif

namespace mhd {
using namespace mhdfft;

template <int N> struct XTeam {
    static constexpr int TP = Plan<N>::TP;
    static constexpr int TEAMS = (TP >= 64) ? 1 : 64 / TP;
    static constexpr int THREADS = TP * TEAMS;
    static constexpr int BUF = Padded::size(N);                 // complex elements per team buffer
    static constexpr size_t SMEM = (size_t)BUF * TEAMS * sizeof(cplx);
};

// product `id` (P_* of mhd_internal.h) at one grid point; inv = 1/rho
__device__ __forceinline__ double product_of(int id, double inv, double mx, double my, double mz, double bx, double by, double bz) {
    switch (id) {
        case P_UX: return mx * inv;
        case P_UY: return my * inv;
        case P_UZ: return mz * inv;
        case P_TXX: return mx * (mx * inv) + 0.5 * (bx * bx + by * by + bz * bz) - bx * bx;
        case P_TYY: return my * (my * inv) + 0.5 * (bx * bx + by * by + bz * bz) - by * by;
        case P_TZZ: return mz * (mz * inv) + 0.5 * (bx * bx + by * by + bz * bz) - bz * bz;
        case P_TXY: return mx * (my * inv) - bx * by;
        case P_TXZ: return mx * (mz * inv) - bx * bz;
        case P_TYZ: return my * (mz * inv) - by * bz;
        case P_EX: return (my * inv) * bz - (mz * inv) * by;
        case P_EY: return (mz * inv) * bx - (mx * inv) * bz;
        case P_EZ: return (mx * inv) * by - (my * inv) * bx;
        default: return 0.0;
    }
}

template <int N, bool HYDRO>
__global__ void __launch_bounds__(XTeam<N>::THREADS, MHD_XFUSED_MINBLOCKS) xfused_kernel(XFusedArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    static_assert(PL::E == 8, "fused x pass needs 8 points per thread");
    constexpr int TP = PL::TP, E = 8;
    constexpr int R0 = PL::radix(0), RL = PL::radix(PL::NP - 1);
    const int team = threadIdx.x / TP, i = threadIdx.x % TP;
    cplx* sm = reinterpret_cast<cplx*>(smraw) + (size_t)team * XTeam<N>::BUF;
    const long long row = (long long)blockIdx.x * XTeam<N>::TEAMS + team;
    const bool ok = row < a.nrows;
    const int nkx = a.nkx;
    cplx* __restrict__ base = a.w2 + row * a.px;
    const Padded lay;

    // 8 grid points x = i + TP*j of: 1/rho, m, B
    // (all seven are initialised: they are filled under a run-time switch inside a rolled loop, and a
    //  value that is undefined on entry lets the compiler fold the conditional stores away)
    double inv[E], mx[E], my[E], mz[E], bx[E], by[E], bz[E];
#pragma unroll
    for (int j = 0; j < E; ++j) { inv[j] = 1.0; mx[j] = 0.0; my[j] = 0.0; mz[j] = 0.0; bx[j] = 0.0; by[j] = 0.0; bz[j] = 0.0; }

    // ---- inverse: field pairs (rho, mx) (my, mz) (Bx, By) (Bz, -) ----
#pragma unroll 1
    for (int pair = 0; pair < (HYDRO ? 2 : 4); ++pair) {
        const cplx* __restrict__ A = base + (long long)(2 * pair) * a.field_stride;
        const cplx* __restrict__ B = A + a.field_stride;
        const bool hasB = pair < 3;
        cplx v[E];
#pragma unroll
        for (int m = 0; m < E / R0; ++m)
#pragma unroll
            for (int q = 0; q < R0; ++q) {
                const int k = first_index<N>(i, m, q);
                cplx z = make_double2(0.0, 0.0);
                if (ok) {
                    if (k < nkx) {
                        cplx x = A[k], y = hasB ? B[k] : make_double2(0.0, 0.0);
                        if (k == 0 || 2 * k == N) { x.y = 0.0; y.y = 0.0; }   // self-conjugate modes: Im ignored
                        z = make_double2(x.x - y.y, x.y + y.x);                // A + iB
                    } else if (N - k < nkx) {
                        cplx x = A[N - k], y = hasB ? B[N - k] : make_double2(0.0, 0.0);
                        z = make_double2(x.x + y.y, y.x - x.y);                // conj(A) + i conj(B)
                    }
                }
                v[m * R0 + q] = z;
            }
        pencil_fft_private<N, true>(v, sm, i, tw);
        const double s = a.scale;
#pragma unroll
        for (int m = 0; m < E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int j = m + q * (E / RL);                 // x = i + TP*j
                const double re = v[m * RL + q].x * s, im = v[m * RL + q].y * s;
                switch (pair) {
                    case 0: inv[j] = re; mx[j] = im; break;
                    case 1: my[j] = re; mz[j] = im; break;
                    case 2: bx[j] = re; by[j] = im; break;
                    default: bz[j] = re; break;
                }
            }
    }
#pragma unroll
    for (int j = 0; j < E; ++j) inv[j] = 1.0 / inv[j];

    // ---- forward: product pairs (ux,uy) (uz,Txx) (Tyy,Tzz) (Txy,Txz) (Tyz,Ex) (Ey,Ez) ----
#pragma unroll 1
    for (int fp = 0; fp < (HYDRO ? 5 : 6); ++fp) {
        int ida, idb;
        switch (fp) {
            case 0: ida = P_UX; idb = P_UY; break;
            case 1: ida = P_UZ; idb = P_TXX; break;
            case 2: ida = P_TYY; idb = P_TZZ; break;
            case 3: ida = P_TXY; idb = P_TXZ; break;
            case 4: ida = P_TYZ; idb = HYDRO ? -1 : P_EX; break;
            default: ida = P_EY; idb = P_EZ; break;
        }
        cplx v[E];
#pragma unroll
        for (int m = 0; m < E / R0; ++m)
#pragma unroll
            for (int q = 0; q < R0; ++q) {
                const int j = m + q * (E / R0);
                v[m * R0 + q] = make_double2(product_of(ida, inv[j], mx[j], my[j], mz[j], bx[j], by[j], bz[j]),
                                             product_of(idb, inv[j], mx[j], my[j], mz[j], bx[j], by[j], bz[j]));
            }
        pencil_fft_private<N, false>(v, sm, i, tw);
        // split Z into the two half-spectra: A[k] = (Z[k] + conj Z[N-k])/2, B[k] = (Z[k] - conj Z[N-k])/(2i)
#pragma unroll
        for (int m = 0; m < E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) sm[lay(last_index<N>(i, m, q))] = v[m * RL + q];
        __syncthreads();
        if (ok) {
            cplx* __restrict__ oa = base + (long long)ida * a.field_stride;
            cplx* __restrict__ ob = base + (long long)(idb < 0 ? 0 : idb) * a.field_stride;
            for (int k = i; k < nkx; k += TP) {
                const cplx zk = sm[lay(k)], zm = sm[lay(k == 0 ? 0 : N - k)];
                oa[k] = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
                if (idb >= 0) ob[k] = make_double2(0.5 * (zk.y + zm.y), 0.5 * (zm.x - zk.x));
            }
        }
        __syncthreads();
    }
}

template <int N> static cudaError_t launch_xfused_n(const XFusedArgs& a, int hydro, const cplx* tw, cudaStream_t st) {
    if constexpr (Plan<N>::E != 8) {
        return cudaErrorInvalidValue;
    } else {
        const unsigned blocks = (unsigned)((a.nrows + XTeam<N>::TEAMS - 1) / XTeam<N>::TEAMS);
        if (hydro) xfused_kernel<N, true><<<blocks, XTeam<N>::THREADS, XTeam<N>::SMEM, st>>>(a, tw);
        else xfused_kernel<N, false><<<blocks, XTeam<N>::THREADS, XTeam<N>::SMEM, st>>>(a, tw);
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
