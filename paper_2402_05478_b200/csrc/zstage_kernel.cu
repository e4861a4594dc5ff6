// zstage_kernel.cu — last forward FFT axis fused with the spectral stage (SURVEY.md §8(a) S3-z + S4):
//
//     12 flux fields on [z][ky][kx]  --z-FFT, pruned to the retained kz-->  i k . , diffusion, forcing,
//     AB2 / RK4 stage update of the 7 state fields,      in ONE pass: the flux spectra G never reach HBM.
//
// eqs (1)-(4) PAPER.md:39-47; "spatial derivative ... 2/3 de-aliasing ... Adams-bashforth" PAPER.md:78.
//
// A CTA owns 8 adjacent (ky,kx) columns (one 128-byte line per z row) and the whole z axis, like the plain
// axis kernel: lane = (column p, slot i), 8 z-outputs per thread.  kx and ky are constant along a column, so the
// right-hand side is assembled by linearity with one or two accumulators per thread instead of 12 live spectra:
//     R_mx = -i [ Z(kx Txx + ky Txy) + kz Z(Txz) ] - nu k^2 Z(ux) - i kx cs^2 rho^ + f^x      (3 transforms)
//     R_my, R_mz alike;   R_rho = -i (kx mx^ + ky my^ + kz mz^) accumulated while m^ is read for its own update;
//     R_Bx = i [ ky Z(Ez) - kz Z(Ey) ],  R_By = i [ kz Z(Ex) - kx Z(Ez) ],  R_Bz = i Z(kx Ey - ky Ex)   (4 transforms)
// 13 transforms per column instead of 12, but 12 spectra less written and read (7.9 GB per step at 512^3).
// With ~120 registers only one 512-thread CTA fits an SM, so the next transform's input tile is fetched with
// cp.async into the thread's own shared-memory slots while the current transform runs (no barrier needed: a
// thread reads back exactly the rows it copied).
#include "mhd_internal.h"
#include "fft_core.cuh"

namespace mhd {
using namespace mhdfft;

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void zs_prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// wavenumber index of FFT index f on an axis of length n
__device__ __forceinline__ int zs_wavenum_full(int f, int n) { return (f < (n + 1) / 2) ? f : f - n; }
// compact (pruned) row of FFT index f when nk rows are stored, or -1
__device__ __forceinline__ int zs_compact(int f, int n, int nk) {
    if (nk == n) return f;
    const int kmax = nk >> 1;
    if (f <= kmax) return f;
    if (f >= n - kmax) return f - (n - nk);
    return -1;
}
__device__ __forceinline__ int zs_wavenum_compact(int j, int nk) { return (j < (nk + 1) / 2) ? j : j - nk; }

// columns per tile: 8 (one 128-byte line per row, one 512-thread CTA per SM at N = 512) or 4 (64-byte segments, two
// 256-thread CTAs per SM).  Measured at 512^3 on B200: 8 -> 4.6 ms, 4 -> 6.1 ms (the 64-byte segments cost more than the
// second CTA gains), so 8 is the default.
#ifndef MHD_ZS_CW
#define MHD_ZS_CW 8
#endif
template <int N> struct ZTile {
    static constexpr int CW = MHD_ZS_CW;
    static constexpr int TP = Plan<N>::TP;
    static constexpr int G = (CW * TP >= 128) ? 1 : 128 / (CW * TP);
    static constexpr int THREADS = CW * TP * G;
    static constexpr int COLS = CW * G;
    static constexpr size_t SMEM = 3 * (size_t)N * COLS * sizeof(cplx);   // exchange + 2 staging tiles
};

// the integrator stage for one mode of one field (same formulas as stage_kernel in mhd_kernels.cu); o = field*F + idx.
// Not inlined: it is called from 5 places x 8 unrolled modes, and the kernel must stay inside the instruction cache.
__device__ __noinline__ void zs_update(cplx* __restrict__ Sp, cplx* __restrict__ Hp, cplx* __restrict__ Ap, long long o, double dt, int mode,
                                       cplx S, cplx R) {
    switch (mode) {
        case STAGE_AB2_EULER: Sp[o] = make_double2(S.x + dt * R.x, S.y + dt * R.y); Hp[o] = R; break;
        case STAGE_AB2: {
            const cplx h = Hp[o];
            Sp[o] = make_double2(S.x + dt * (1.5 * R.x - 0.5 * h.x), S.y + dt * (1.5 * R.y - 0.5 * h.y));
            Hp[o] = R;
        } break;
        case STAGE_RK4_1:
            Hp[o] = S;
            Ap[o] = make_double2(S.x + dt / 6.0 * R.x, S.y + dt / 6.0 * R.y);
            Sp[o] = make_double2(S.x + 0.5 * dt * R.x, S.y + 0.5 * dt * R.y);
            break;
        case STAGE_RK4_2: {
            const cplx ac = Ap[o], h = Hp[o];
            Ap[o] = make_double2(ac.x + dt / 3.0 * R.x, ac.y + dt / 3.0 * R.y);
            Sp[o] = make_double2(h.x + 0.5 * dt * R.x, h.y + 0.5 * dt * R.y);
        } break;
        case STAGE_RK4_3: {
            const cplx ac = Ap[o], h = Hp[o];
            Ap[o] = make_double2(ac.x + dt / 3.0 * R.x, ac.y + dt / 3.0 * R.y);
            Sp[o] = make_double2(h.x + dt * R.x, h.y + dt * R.y);
        } break;
        default: {
            const cplx ac = Ap[o];
            Sp[o] = make_double2(ac.x + dt / 6.0 * R.x, ac.y + dt / 6.0 * R.y);
        } break;
    }
}

// steady-state AB2 (the hot case): inlined, so the compiler can batch the eight history loads of a finish phase
__device__ __forceinline__ void zs_update_ab2(cplx* __restrict__ Sp, cplx* __restrict__ Hp, long long o, double dt, cplx S, cplx R) {
    const cplx h = Hp[o];
    Sp[o] = make_double2(S.x + dt * (1.5 * R.x - 0.5 * h.x), S.y + dt * (1.5 * R.y - 0.5 * h.y));
    Hp[o] = R;
}

// AB2STEADY: the stage is known at compile time to be STAGE_AB2
template <int N, bool HYDRO, bool AB2STEADY>
__global__ void __launch_bounds__(ZTile<N>::THREADS, (ZTile<N>::CW == 4 && ZTile<N>::THREADS <= 256) ? 2 : 1) zstage_kernel(ZStageArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    static_assert(PL::E == 8 && PL::radix(0) == 8, "zstage needs 8 points per thread and a radix-8 first pass");
    constexpr int TP = PL::TP, E = 8, RL = PL::radix(PL::NP - 1);
    constexpr int G = ZTile<N>::G, CW = ZTile<N>::CW;
    const int tid = threadIdx.x, p = tid & (CW - 1), i = (tid / CW) % TP, g = tid / (CW * TP);
    cplx* const ex = reinterpret_cast<cplx*>(smraw) + (size_t)g * N * CW;
    cplx* const st0 = reinterpret_cast<cplx*>(smraw) + (size_t)(G + g) * N * CW;
    cplx* const st1 = st0 + (size_t)G * N * CW;
    const StageArgs& s = a.st;
    const SpecGeom& geo = s.g;
    const long long F = geo.field;
    const long long col = (long long)blockIdx.x * ZTile<N>::COLS + g * CW + p;
    const int jx = (int)(col % geo.px);
    const int jy = (int)(col / geo.px);
    const bool colok = col < a.inner && jx < geo.nkx;
    const double kx = s.kfx * (double)jx, ky = s.kfy * (double)zs_wavenum_compact(jy, geo.nky);
    const double kxy2 = kx * kx + ky * ky;

    // ---- staging: each thread copies (cp.async) and later reads back its own 8 rows of a tile ----
    auto issue = [&](int field, cplx* buf) {
        if (colok && field >= 0) {
            const cplx* src = a.W1 + (long long)field * a.w1field + col;
#pragma unroll
            for (int q = 0; q < E; ++q) cp_async16(&buf[(i + TP * q) * CW + p], src + (long long)(i + TP * q) * a.inner);
        }
        cp_async_commit();
    };
    // output register r = m*RL + q holds FFT index f(r); kz and the compact state index follow from it
    auto out_index = [&](int m, int q, double& kz, long long& idx) -> bool {
        const int f = last_index<N>(i, m, q);
        const int c = zs_compact(f, N, geo.nkz);
        kz = s.kfz * (double)zs_wavenum_full(f, N);
        idx = (long long)c * a.inner + col;
        return colok && c >= 0;
    };
    // pull the state / history lines this thread will touch in a finish phase into L2 ahead of time (no registers)
    auto prefetch_state = [&](int field) {
        if (!colok || p != 0) return;            // one lane per tile row (a 128- or 64-byte segment)
#pragma unroll
        for (int m = 0; m < E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                double kz; long long idx;
                if (!out_index(m, q, kz, idx)) continue;
                zs_prefetch_l2(&s.S[(long long)field * F + idx]);
                if (AB2STEADY || (s.mode != STAGE_AB2_EULER && s.mode != STAGE_RK4_1)) zs_prefetch_l2(&s.H[(long long)field * F + idx]);
                if (!AB2STEADY && s.mode >= STAGE_RK4_2) zs_prefetch_l2(&s.Acc[(long long)field * F + idx]);
            }
    };

    cplx v[E], acc[E], rr[E];
#pragma unroll
    for (int r = 0; r < E; ++r) { rr[r] = make_double2(0.0, 0.0); acc[r] = make_double2(0.0, 0.0); }

    // Job list (one z transform each).  Momentum component c = 0,1,2 takes jobs 3c..3c+2:
    //   3c   : Z(kx T_cx + ky T_cy)          -> acc
    //   3c+1 : Z(T_cz)                       -> acc += kz * .
    //   3c+2 : Z(u_c)                        -> update m_c; after c = 2 also rho
    // induction: 9: Z(Ex) -> aby = kz .;  10: Z(Ey) -> abx = -kz .;  11: Z(Ez) -> update Bx, By;  12: Z(kx Ey - ky Ex) -> update Bz
    constexpr int NJOB = HYDRO ? 9 : 13;
    issue(P_TXX, st0);
    issue(P_TXY, st1);
    prefetch_state(F_RHO);
#pragma unroll 1
    for (int j = 0; j < NJOB; ++j) {
        const int c = j / 3, ph = j - 3 * c;
        // ---- fetch this job's input from the staging slots ----
        cp_async_wait_all();
        if (j < 9 ? ph == 0 : j == 12) {
            const double ca = (j == 12) ? -ky : kx, cb = (j == 12) ? kx : ky;      // job 12: st0 = Ex, st1 = Ey
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const cplx x = colok ? st0[(i + TP * q) * CW + p] : make_double2(0.0, 0.0);
                const cplx y = colok ? st1[(i + TP * q) * CW + p] : make_double2(0.0, 0.0);
                v[q] = make_double2(ca * x.x + cb * y.x, ca * x.y + cb * y.y);
            }
        } else {
            const cplx* buf = (j < 9 ? ph == 1 : (j != 10)) ? st0 : st1;
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = colok ? buf[(i + TP * q) * CW + p] : make_double2(0.0, 0.0);
        }
        // ---- refill the slots just read with the tiles of the next jobs ----
        {
            int f0 = -1, f1 = -1;
            if (j < 9) {
                if (ph == 0) { f0 = (c == 0) ? P_TXZ : (c == 1) ? P_TYZ : P_TZZ; f1 = P_UX + c; }
                else if (ph == 1) f0 = (c == 0) ? P_TXY : (c == 1) ? P_TXZ : (HYDRO ? -1 : P_EX);
                else f1 = (c == 0) ? P_TYY : (c == 1) ? P_TYZ : (HYDRO ? -1 : P_EY);
            } else if (j == 9) f0 = P_EZ;
            else if (j == 10) f1 = P_EY;
            else if (j == 11) f0 = P_EX;
            if (f0 >= 0) issue(f0, st0);
            if (f1 >= 0) issue(f1, st1);
            // the state lines the job after next will update
            if (j < 9 && ph == 1) prefetch_state(F_MX + c);
            if (j == 9) { prefetch_state(F_BX); prefetch_state(F_BY); }
            if (j == 11) prefetch_state(F_BZ);
        }
        if constexpr (CW == 8) pencil_fft<N, false>(v, ex, i, p, tw);
        else pencil_fft4<N, false>(v, ex, i, p, tw);
        // ---- consume ----
#pragma unroll
        for (int m = 0; m < E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int r = m * RL + q;
                double kz; long long idx;
                const bool ok = out_index(m, q, kz, idx);
                if (j < 9 && ph == 0) { acc[r] = v[r]; continue; }
                if (j < 9 && ph == 1) { acc[r].x += kz * v[r].x; acc[r].y += kz * v[r].y; continue; }
                if (j == 9) { rr[r] = make_double2(kz * v[r].x, kz * v[r].y); continue; }        // aby = kz Ex
                if (j == 10) { acc[r] = make_double2(-kz * v[r].x, -kz * v[r].y); continue; }    // abx = -kz Ey
                if (!ok) continue;
                const double k2 = kxy2 + kz * kz;
                if (j < 9) {                     // eqs (2), (3): R_m,c = -i D - nu k^2 u^_c - i k_c cs^2 rho^ + f^_c
                    const double vk = s.nu * k2;
                    const double kc = (c == 0) ? kx : (c == 1) ? ky : kz;
                    const cplx rho = s.S[F_RHO * F + idx], mc = s.S[(long long)(F_MX + c) * F + idx];
                    const double pk = kc * s.cs2;
                    cplx R = make_double2(acc[r].y - vk * v[r].x + pk * rho.y, -acc[r].x - vk * v[r].y - pk * rho.x);
                    if (s.F) { const cplx f = s.F[(long long)c * F + idx]; R.x += f.x; R.y += f.y; }
                    rr[r].x += kc * mc.x; rr[r].y += kc * mc.y;
                    { if constexpr (AB2STEADY) zs_update_ab2(s.S, s.H, (long long)(F_MX + c) * F + idx, s.dt, mc, R); else zs_update(s.S, s.H, s.Acc, (long long)(F_MX + c) * F + idx, s.dt, s.mode, mc, R); }
                    if (c == 2) { if constexpr (AB2STEADY) zs_update_ab2(s.S, s.H, (long long)(F_RHO) * F + idx, s.dt, rho, make_double2(rr[r].y, -rr[r].x)); else zs_update(s.S, s.H, s.Acc, (long long)(F_RHO) * F + idx, s.dt, s.mode, rho, make_double2(rr[r].y, -rr[r].x)); }   // eq. (1): R_rho = -i k.m^
                } else if (j == 11) {            // eq. (4): R_Bx = i (ky Ez - kz Ey), R_By = i (kz Ex - kx Ez), - eta k^2 B^
                    const double ek = s.eta * k2;
                    const cplx cx = make_double2(acc[r].x + ky * v[r].x, acc[r].y + ky * v[r].y);
                    const cplx cy = make_double2(rr[r].x - kx * v[r].x, rr[r].y - kx * v[r].y);
                    const cplx bx = s.S[F_BX * F + idx], by = s.S[F_BY * F + idx];
                    { if constexpr (AB2STEADY) zs_update_ab2(s.S, s.H, (long long)(F_BX) * F + idx, s.dt, bx, make_double2(-cx.y - ek * bx.x, cx.x - ek * bx.y)); else zs_update(s.S, s.H, s.Acc, (long long)(F_BX) * F + idx, s.dt, s.mode, bx, make_double2(-cx.y - ek * bx.x, cx.x - ek * bx.y)); }
                    { if constexpr (AB2STEADY) zs_update_ab2(s.S, s.H, (long long)(F_BY) * F + idx, s.dt, by, make_double2(-cy.y - ek * by.x, cy.x - ek * by.y)); else zs_update(s.S, s.H, s.Acc, (long long)(F_BY) * F + idx, s.dt, s.mode, by, make_double2(-cy.y - ek * by.x, cy.x - ek * by.y)); }
                } else {                         // j == 12: R_Bz = i (kx Ey - ky Ex) - eta k^2 Bz^
                    const double ek = s.eta * k2;
                    const cplx bz = s.S[F_BZ * F + idx];
                    { if constexpr (AB2STEADY) zs_update_ab2(s.S, s.H, (long long)(F_BZ) * F + idx, s.dt, bz, make_double2(-v[r].y - ek * bz.x, v[r].x - ek * bz.y)); else zs_update(s.S, s.H, s.Acc, (long long)(F_BZ) * F + idx, s.dt, s.mode, bz, make_double2(-v[r].y - ek * bz.x, v[r].x - ek * bz.y)); }
                }
            }
    }
}

template <int N> static cudaError_t launch_zstage_n(const ZStageArgs& a, const cplx* tw, cudaStream_t st) {
    if constexpr (Plan<N>::E != 8 || N > 512) {
        return cudaErrorInvalidValue;
    } else {
        static DeviceOnce once;
        const int dev = device_slot();
        if (dev < 0) return cudaErrorInvalidDevice;
        if (!once.done[dev]) {
            cudaError_t e = cudaFuncSetAttribute(zstage_kernel<N, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZTile<N>::SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(zstage_kernel<N, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZTile<N>::SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(zstage_kernel<N, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZTile<N>::SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(zstage_kernel<N, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZTile<N>::SMEM);
            if (e != cudaSuccess) return e;
            once.done[dev] = true;
        }
        const unsigned blocks = (unsigned)((a.inner + ZTile<N>::COLS - 1) / ZTile<N>::COLS);
        if (a.st.mode == STAGE_AB2) {
            if (a.st.hydro) zstage_kernel<N, true, true><<<blocks, ZTile<N>::THREADS, ZTile<N>::SMEM, st>>>(a, tw);
            else zstage_kernel<N, false, true><<<blocks, ZTile<N>::THREADS, ZTile<N>::SMEM, st>>>(a, tw);
        } else {
            if (a.st.hydro) zstage_kernel<N, true, false><<<blocks, ZTile<N>::THREADS, ZTile<N>::SMEM, st>>>(a, tw);
            else zstage_kernel<N, false, false><<<blocks, ZTile<N>::THREADS, ZTile<N>::SMEM, st>>>(a, tw);
        }
        count_launch();
        return cudaGetLastError();
    }
}

bool zstage_supported(int n) {
    switch (n) {
        case 8: case 16: case 32: case 64: case 128: case 256: case 512: return true;
        default: return false;
    }
}

cudaError_t launch_zstage(int n, const ZStageArgs& a, const double2* tw, cudaStream_t st) {
    switch (n) {
        case 8: return launch_zstage_n<8>(a, tw, st);
        case 16: return launch_zstage_n<16>(a, tw, st);
        case 32: return launch_zstage_n<32>(a, tw, st);
        case 64: return launch_zstage_n<64>(a, tw, st);
        case 128: return launch_zstage_n<128>(a, tw, st);
        case 256: return launch_zstage_n<256>(a, tw, st);
        case 512: return launch_zstage_n<512>(a, tw, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace mhd
