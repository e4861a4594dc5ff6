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

template <int N> struct ZTile {
    static constexpr int TP = Plan<N>::TP;
    static constexpr int G = Tile<N>::G;
    static constexpr int THREADS = Tile<N>::THREADS;
    static constexpr int COLS = Tile<N>::COLS;
    static constexpr size_t SMEM = 3 * (size_t)N * COLS * sizeof(cplx);   // exchange + 2 staging tiles
};

// the integrator stage for one mode of one field (same formulas as stage_kernel in mhd_kernels.cu)
__device__ __forceinline__ void zs_update(const StageArgs& a, int f, long long idx, cplx S, cplx R) {
    const long long o = (long long)f * a.g.field + idx;
    const double dt = a.dt;
    switch (a.mode) {
        case STAGE_AB2_EULER: a.S[o] = make_double2(S.x + dt * R.x, S.y + dt * R.y); a.H[o] = R; break;
        case STAGE_AB2: {
            const cplx h = a.H[o];
            a.S[o] = make_double2(S.x + dt * (1.5 * R.x - 0.5 * h.x), S.y + dt * (1.5 * R.y - 0.5 * h.y));
            a.H[o] = R;
        } break;
        case STAGE_RK4_1:
            a.H[o] = S;
            a.Acc[o] = make_double2(S.x + dt / 6.0 * R.x, S.y + dt / 6.0 * R.y);
            a.S[o] = make_double2(S.x + 0.5 * dt * R.x, S.y + 0.5 * dt * R.y);
            break;
        case STAGE_RK4_2: {
            const cplx ac = a.Acc[o], h = a.H[o];
            a.Acc[o] = make_double2(ac.x + dt / 3.0 * R.x, ac.y + dt / 3.0 * R.y);
            a.S[o] = make_double2(h.x + 0.5 * dt * R.x, h.y + 0.5 * dt * R.y);
        } break;
        case STAGE_RK4_3: {
            const cplx ac = a.Acc[o], h = a.H[o];
            a.Acc[o] = make_double2(ac.x + dt / 3.0 * R.x, ac.y + dt / 3.0 * R.y);
            a.S[o] = make_double2(h.x + dt * R.x, h.y + dt * R.y);
        } break;
        default: {
            const cplx ac = a.Acc[o];
            a.S[o] = make_double2(ac.x + dt / 6.0 * R.x, ac.y + dt / 6.0 * R.y);
        } break;
    }
}

template <int N, bool HYDRO>
__global__ void __launch_bounds__(ZTile<N>::THREADS, 1) zstage_kernel(ZStageArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    static_assert(PL::E == 8 && PL::radix(0) == 8, "zstage needs 8 points per thread and a radix-8 first pass");
    constexpr int TP = PL::TP, E = 8, RL = PL::radix(PL::NP - 1);
    constexpr int G = ZTile<N>::G;
    const int tid = threadIdx.x, p = tid & 7, i = (tid >> 3) % TP, g = tid / (8 * TP);
    cplx* const ex = reinterpret_cast<cplx*>(smraw) + (size_t)g * N * 8;
    cplx* const st0 = reinterpret_cast<cplx*>(smraw) + (size_t)(G + g) * N * 8;
    cplx* const st1 = st0 + (size_t)G * N * 8;
    const StageArgs& s = a.st;
    const SpecGeom& geo = s.g;
    const long long F = geo.field;
    const long long col = (long long)blockIdx.x * ZTile<N>::COLS + g * 8 + p;
    const int jx = (int)(col % geo.px);
    const int jy = (int)(col / geo.px);
    const bool colok = col < a.inner && jx < geo.nkx;
    const double kx = s.kfx * (double)jx, ky = s.kfy * (double)zs_wavenum_compact(jy, geo.nky);
    const double kxy2 = kx * kx + ky * ky;

    // ---- staging: each thread copies (cp.async) and later reads back its own 8 rows of a tile ----
    auto issue = [&](int field, cplx* buf) {
        if (colok) {
            const cplx* src = a.W1 + (long long)field * a.w1field + col;
#pragma unroll
            for (int q = 0; q < E; ++q) cp_async16(&buf[(i + TP * q) * 8 + p], src + (long long)(i + TP * q) * a.inner);
        }
        cp_async_commit();
    };
    auto fetch1 = [&](cplx (&v)[E], const cplx* buf) {
        cp_async_wait_all();
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = colok ? buf[(i + TP * q) * 8 + p] : make_double2(0.0, 0.0);
    };
    auto fetch2 = [&](cplx (&v)[E], const cplx* ba, double ca, const cplx* bb, double cb) {   // ca*A + cb*B
        cp_async_wait_all();
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const cplx x = colok ? ba[(i + TP * q) * 8 + p] : make_double2(0.0, 0.0);
            const cplx y = colok ? bb[(i + TP * q) * 8 + p] : make_double2(0.0, 0.0);
            v[q] = make_double2(ca * x.x + cb * y.x, ca * x.y + cb * y.y);
        }
    };
    // output register r = m*RL + q holds FFT index f(r); kz and the compact state index follow from it
    auto out_index = [&](int m, int q, double& kz, long long& idx) -> bool {
        const int f = last_index<N>(i, m, q);
        const int c = zs_compact(f, N, geo.nkz);
        kz = s.kfz * (double)zs_wavenum_full(f, N);
        idx = (long long)c * a.inner + col;
        return colok && c >= 0;
    };

    cplx v[E], acc[E], rr[E];
#pragma unroll
    for (int r = 0; r < E; ++r) rr[r] = make_double2(0.0, 0.0);

    // momentum component c: D = kx T_cx + ky T_cy + kz T_cz (accumulated), U = u_c
    auto finish_momentum = [&](int c) {
#pragma unroll
        for (int m = 0; m < E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int r = m * RL + q;
                double kz; long long idx;
                if (!out_index(m, q, kz, idx)) continue;
                const double k2 = kxy2 + kz * kz, vk = s.nu * k2;
                const double kc = (c == 0) ? kx : (c == 1) ? ky : kz;
                const cplx rho = s.S[F_RHO * F + idx], mc = s.S[(F_MX + c) * F + idx];
                const double pk = kc * s.cs2;
                cplx R = make_double2(acc[r].y - vk * v[r].x + pk * rho.y, -acc[r].x - vk * v[r].y - pk * rho.x);
                if (s.F) { const cplx f = s.F[c * F + idx]; R.x += f.x; R.y += f.y; }
                rr[r].x += kc * mc.x; rr[r].y += kc * mc.y;
                zs_update(s, F_MX + c, idx, mc, R);
            }
    };

    // ---- momentum (eqs 2, 3) and, from the m^ read on the way, continuity (eq. 1) ----
    constexpr int CA[3] = {P_TXX, P_TXY, P_TXZ};     // multiplied by kx
    constexpr int CB[3] = {P_TXY, P_TYY, P_TYZ};     // multiplied by ky
    constexpr int CC[3] = {P_TXZ, P_TYZ, P_TZZ};     // multiplied by kz (after the transform)
    constexpr int CU[3] = {P_UX, P_UY, P_UZ};
    issue(CA[0], st0);
    issue(CB[0], st1);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // job 1: Z(kx T_cx + ky T_cy)
        fetch2(v, st0, kx, st1, ky);
        issue(CC[c], st0);
        issue(CU[c], st1);
        pencil_fft<N, false>(v, ex, i, p, tw);
#pragma unroll
        for (int r = 0; r < E; ++r) acc[r] = v[r];
        // job 2: + kz Z(T_cz)
        fetch1(v, st0);
        if (c < 2) issue(CA[c + 1], st0);
        else if (!HYDRO) issue(P_EX, st0);
        pencil_fft<N, false>(v, ex, i, p, tw);
#pragma unroll
        for (int m = 0; m < E / RL; ++m)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int r = m * RL + q;
                const double kz = s.kfz * (double)zs_wavenum_full(last_index<N>(i, m, q), N);
                acc[r].x += kz * v[r].x; acc[r].y += kz * v[r].y;
            }
        // job 3: Z(u_c), then the update of m_c
        fetch1(v, st1);
        if (c < 2) issue(CB[c + 1], st1);
        else if (!HYDRO) issue(P_EY, st1);
        pencil_fft<N, false>(v, ex, i, p, tw);
        finish_momentum(c);
    }
    // continuity: R_rho = -i k.m^
#pragma unroll
    for (int m = 0; m < E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int r = m * RL + q;
            double kz; long long idx;
            if (!out_index(m, q, kz, idx)) continue;
            zs_update(s, F_RHO, idx, s.S[F_RHO * F + idx], make_double2(rr[r].y, -rr[r].x));
        }
    if constexpr (HYDRO) return;

    // ---- induction (eq. 4): R_B = i k x E^ - eta k^2 B^ ----
    cplx (&abx)[E] = acc;      // ky Ez - kz Ey
    cplx (&aby)[E] = rr;       // kz Ex - kx Ez
    fetch1(v, st0);            // Ex
    issue(P_EZ, st0);
    pencil_fft<N, false>(v, ex, i, p, tw);
#pragma unroll
    for (int m = 0; m < E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int r = m * RL + q;
            const double kz = s.kfz * (double)zs_wavenum_full(last_index<N>(i, m, q), N);
            aby[r] = make_double2(kz * v[r].x, kz * v[r].y);
        }
    fetch1(v, st1);            // Ey
    issue(P_EY, st1);
    pencil_fft<N, false>(v, ex, i, p, tw);
#pragma unroll
    for (int m = 0; m < E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int r = m * RL + q;
            const double kz = s.kfz * (double)zs_wavenum_full(last_index<N>(i, m, q), N);
            abx[r] = make_double2(-kz * v[r].x, -kz * v[r].y);
        }
    fetch1(v, st0);            // Ez
    issue(P_EX, st0);
    pencil_fft<N, false>(v, ex, i, p, tw);
#pragma unroll
    for (int m = 0; m < E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int r = m * RL + q;
            double kz; long long idx;
            if (!out_index(m, q, kz, idx)) continue;
            const double ek = s.eta * (kxy2 + kz * kz);
            const cplx cx = make_double2(abx[r].x + ky * v[r].x, abx[r].y + ky * v[r].y);
            const cplx cy = make_double2(aby[r].x - kx * v[r].x, aby[r].y - kx * v[r].y);
            const cplx bx = s.S[F_BX * F + idx], by = s.S[F_BY * F + idx];
            zs_update(s, F_BX, idx, bx, make_double2(-cx.y - ek * bx.x, cx.x - ek * bx.y));
            zs_update(s, F_BY, idx, by, make_double2(-cy.y - ek * by.x, cy.x - ek * by.y));
        }
    fetch2(v, st1, kx, st0, -ky);     // kx Ey - ky Ex
    pencil_fft<N, false>(v, ex, i, p, tw);
#pragma unroll
    for (int m = 0; m < E / RL; ++m)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int r = m * RL + q;
            double kz; long long idx;
            if (!out_index(m, q, kz, idx)) continue;
            const double ek = s.eta * (kxy2 + kz * kz);
            const cplx bz = s.S[F_BZ * F + idx];
            zs_update(s, F_BZ, idx, bz, make_double2(-v[r].y - ek * bz.x, v[r].x - ek * bz.y));
        }
}

template <int N> static cudaError_t launch_zstage_n(const ZStageArgs& a, const cplx* tw, cudaStream_t st) {
    if constexpr (Plan<N>::E != 8 || N > 512) {
        return cudaErrorInvalidValue;
    } else {
        static bool attr_done = false;
        if (!attr_done) {
            cudaError_t e = cudaFuncSetAttribute(zstage_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZTile<N>::SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(zstage_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZTile<N>::SMEM);
            if (e != cudaSuccess) return e;
            attr_done = true;
        }
        const unsigned blocks = (unsigned)((a.inner + ZTile<N>::COLS - 1) / ZTile<N>::COLS);
        if (a.st.hydro) zstage_kernel<N, true><<<blocks, ZTile<N>::THREADS, ZTile<N>::SMEM, st>>>(a, tw);
        else zstage_kernel<N, false><<<blocks, ZTile<N>::THREADS, ZTile<N>::SMEM, st>>>(a, tw);
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
