// mhd_kernels.cu — real-space products (S2), spectral stage update (S4) and diagnostics reductions
// (S5) of the pseudo-spectral MHD step (eqs (1)-(4) PAPER.md:39-47).
#include "mhd_internal.h"

#include <atomic>

namespace mhd {

static std::atomic<long long> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }
long long launch_count() { return g_launches.load(std::memory_order_relaxed); }
void add_launches(long long n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int device_slot() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return -1;
    return dev;
}
cudaError_t device_sm_count(int dev, int* sms) {
    static int cache[kMaxDevices];           // 0 = not asked yet (benign race: every writer stores the same value)
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    if (cache[dev] == 0) {
        int v = 0;
        cudaError_t e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        cache[dev] = v;
    }
    *sms = cache[dev];
    return cudaSuccess;
}

static constexpr int kThreads = 256;
static constexpr int kGridStream = 148 * 8;   // grid-stride kernels: 8 CTAs of 256 threads per SM

// ---- S2: products ----------------------------------------------------------------------------
// in : rho, m, B on the grid (7 consecutive fields, or 4 when hydro)
// out: u (3), T_xx T_yy T_zz T_xy T_xz T_yz (6), E = u x B (3; skipped when hydro)
//      T_ij = m_i u_j + delta_ij |B|^2/2 - B_i B_j     (eq. 2: rho u u + (B^2/2) I - B B; the
//      isothermal pressure Cs^2 rho is linear and is added spectrally in the stage kernel)
template <bool HYDRO>
__global__ void __launch_bounds__(kThreads) products_kernel(const double* __restrict__ f, double* __restrict__ g, long long npts) {
    const long long n2 = npts >> 1;   // nx is even: process double2
    const double2* __restrict__ f2 = reinterpret_cast<const double2*>(f);
    double2* __restrict__ g2 = reinterpret_cast<double2*>(g);
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n2; idx += (long long)gridDim.x * blockDim.x) {
        const double2 rho = f2[F_RHO * n2 + idx], mx = f2[F_MX * n2 + idx], my = f2[F_MY * n2 + idx], mz = f2[F_MZ * n2 + idx];
        double2 bx = make_double2(0, 0), by = bx, bz = bx;
        if (!HYDRO) { bx = f2[F_BX * n2 + idx]; by = f2[F_BY * n2 + idx]; bz = f2[F_BZ * n2 + idx]; }
        double out[NPROD][2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double r = h ? rho.y : rho.x;
            const double Mx = h ? mx.y : mx.x, My = h ? my.y : my.x, Mz = h ? mz.y : mz.x;
            const double Bx = h ? bx.y : bx.x, By = h ? by.y : by.x, Bz = h ? bz.y : bz.x;
            const double inv = 1.0 / r;
            const double ux = Mx * inv, uy = My * inv, uz = Mz * inv;
            const double b2h = 0.5 * (Bx * Bx + By * By + Bz * Bz);
            out[P_UX][h] = ux; out[P_UY][h] = uy; out[P_UZ][h] = uz;
            out[P_TXX][h] = Mx * ux + b2h - Bx * Bx;
            out[P_TYY][h] = My * uy + b2h - By * By;
            out[P_TZZ][h] = Mz * uz + b2h - Bz * Bz;
            out[P_TXY][h] = Mx * uy - Bx * By;
            out[P_TXZ][h] = Mx * uz - Bx * Bz;
            out[P_TYZ][h] = My * uz - By * Bz;
            out[P_EX][h] = uy * Bz - uz * By;
            out[P_EY][h] = uz * Bx - ux * Bz;
            out[P_EZ][h] = ux * By - uy * Bx;
        }
#pragma unroll
        for (int j = 0; j < (HYDRO ? P_EX : NPROD); ++j) g2[(long long)j * n2 + idx] = make_double2(out[j][0], out[j][1]);
    }
}

cudaError_t launch_products(const double* f, double* g, long long npts, int hydro, cudaStream_t st) {
    if (hydro) products_kernel<true><<<kGridStream, kThreads, 0, st>>>(f, g, npts);
    else products_kernel<false><<<kGridStream, kThreads, 0, st>>>(f, g, npts);
    count_launch();
    return cudaGetLastError();
}

// ---- small pointwise helpers -----------------------------------------------------------------
__global__ void momentum_kernel(const double* __restrict__ rho, const double* __restrict__ ux, const double* __restrict__ uy,
                                const double* __restrict__ uz, double* __restrict__ m, long long npts) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < npts; i += (long long)gridDim.x * blockDim.x) {
        const double r = rho[i];
        m[i] = r * ux[i]; m[npts + i] = r * uy[i]; m[2 * npts + i] = r * uz[i];
    }
}
cudaError_t launch_momentum(const double* rho, const double* ux, const double* uy, const double* uz, double* m,
                            long long npts, cudaStream_t st) {
    momentum_kernel<<<kGridStream, kThreads, 0, st>>>(rho, ux, uy, uz, m, npts);
    count_launch();
    return cudaGetLastError();
}

__global__ void velocity_kernel(const double* __restrict__ f, double* __restrict__ ux, double* __restrict__ uy,
                                double* __restrict__ uz, long long npts) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < npts; i += (long long)gridDim.x * blockDim.x) {
        const double r = f[F_RHO * npts + i];
        ux[i] = f[F_MX * npts + i] / r; uy[i] = f[F_MY * npts + i] / r; uz[i] = f[F_MZ * npts + i] / r;
    }
}
cudaError_t launch_velocity(const double* f, double* ux, double* uy, double* uz, long long npts, cudaStream_t st) {
    velocity_kernel<<<kGridStream, kThreads, 0, st>>>(f, ux, uy, uz, npts);
    count_launch();
    return cudaGetLastError();
}
cudaError_t launch_velocity3(const double* f, double* u3, long long npts, cudaStream_t st) {
    return launch_velocity(f, u3, u3 + npts, u3 + 2 * npts, npts, st);
}

cudaError_t launch_zero(void* p, size_t bytes, cudaStream_t st) { return cudaMemsetAsync(p, 0, bytes, st); }

// ---- S4: spectral assembly + diffusion + time-integrator stage ---------------------------------
// wavenumber of stored index j on an axis storing nk modes in FFT order (nk = n or 2*kmax+1)
__device__ __forceinline__ double wavenum(int j, int nk) { return (double)((j < (nk + 1) / 2) ? j : j - nk); }

__device__ __forceinline__ double2 axpy(double2 a, double s, double2 r) { return make_double2(a.x + s * r.x, a.y + s * r.y); }

#ifndef MHD_STAGE_SPLIT
#define MHD_STAGE_SPLIT 1      // 1: the MHD stage runs as two launches, (rho, m) then B: fewer concurrent streams per kernel
#endif
// PART 0: all seven fields; 1: rho and m only (the whole stage of a hydrodynamic run); 2: B only
template <int PART>
__global__ void __launch_bounds__(kThreads) stage_kernel(StageArgs a) {
    constexpr bool HYDRO = (PART == 1);
    constexpr int F0 = (PART == 2) ? F_BX : 0, F1 = (PART == 1) ? 4 : NFIELD;
    const SpecGeom g = a.g;
    const long long total = g.field;
    const long long F = g.field;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const int jx = (int)(idx % g.px);
        if (jx >= g.nkx) continue;
        const long long row = idx / g.px;
        const int jy = (int)(row % g.nky), jz = (int)(row / g.nky);
        const double kx = a.kfx * (double)jx, ky = a.kfy * wavenum(jy, g.nky), kz = a.kfz * wavenum(jz, g.nkz);
        const double k2 = kx * kx + ky * ky + kz * kz;

        double2 S[NFIELD], R[NFIELD];
#pragma unroll
        for (int f = F0; f < F1; ++f) S[f] = a.S[f * F + idx];
        const double2* __restrict__ G = a.G + idx;
        // eq. (1): R_rho = -i k.m^
        if (PART != 2) {
            const double dx = kx * S[F_MX].x + ky * S[F_MY].x + kz * S[F_MZ].x;
            const double dy = kx * S[F_MX].y + ky * S[F_MY].y + kz * S[F_MZ].y;
            R[F_RHO] = make_double2(dy, -dx);
        }
        // eqs (2)+(3): R_m,i = -i k_j T^_ij - i k_i cs^2 rho^ - nu k^2 u^_i
        if (PART != 2) {
            const double2 txx = G[P_TXX * F], tyy = G[P_TYY * F], tzz = G[P_TZZ * F];
            const double2 txy = G[P_TXY * F], txz = G[P_TXZ * F], tyz = G[P_TYZ * F];
            const double2 ux = G[P_UX * F], uy = G[P_UY * F], uz = G[P_UZ * F];
            const double2 pr = make_double2(a.cs2 * S[F_RHO].x, a.cs2 * S[F_RHO].y);
            const double vk = a.nu * k2;
            double dx, dy;
            dx = kx * (txx.x + pr.x) + ky * txy.x + kz * txz.x; dy = kx * (txx.y + pr.y) + ky * txy.y + kz * txz.y;
            R[F_MX] = make_double2(dy - vk * ux.x, -dx - vk * ux.y);
            dx = kx * txy.x + ky * (tyy.x + pr.x) + kz * tyz.x; dy = kx * txy.y + ky * (tyy.y + pr.y) + kz * tyz.y;
            R[F_MY] = make_double2(dy - vk * uy.x, -dx - vk * uy.y);
            dx = kx * txz.x + ky * tyz.x + kz * (tzz.x + pr.x); dy = kx * txz.y + ky * tyz.y + kz * (tzz.y + pr.y);
            R[F_MZ] = make_double2(dy - vk * uz.x, -dx - vk * uz.y);
            if (a.F) {   // eq. (2): + f (steady body force; stored pruned, i.e. already masked)
                const double2 fx = a.F[idx], fy = a.F[F + idx], fz = a.F[2 * F + idx];
                R[F_MX].x += fx.x; R[F_MX].y += fx.y; R[F_MY].x += fy.x; R[F_MY].y += fy.y; R[F_MZ].x += fz.x; R[F_MZ].y += fz.y;
            }
        }
        // eq. (4): R_B = i k x E^ - eta k^2 B^
        if (!HYDRO) {
            const double2 ex = G[P_EX * F], ey = G[P_EY * F], ez = G[P_EZ * F];
            const double ek = a.eta * k2;
            double cx, cy;
            cx = ky * ez.x - kz * ey.x; cy = ky * ez.y - kz * ey.y;
            R[F_BX] = make_double2(-cy - ek * S[F_BX].x, cx - ek * S[F_BX].y);
            cx = kz * ex.x - kx * ez.x; cy = kz * ex.y - kx * ez.y;
            R[F_BY] = make_double2(-cy - ek * S[F_BY].x, cx - ek * S[F_BY].y);
            cx = kx * ey.x - ky * ex.x; cy = kx * ey.y - ky * ex.y;
            R[F_BZ] = make_double2(-cy - ek * S[F_BZ].x, cx - ek * S[F_BZ].y);
        }
        const double dt = a.dt;
#pragma unroll
        for (int f = F0; f < F1; ++f) {
            const long long o = f * F + idx;
            switch (a.mode) {
                case STAGE_AB2_EULER: a.S[o] = axpy(S[f], dt, R[f]); a.H[o] = R[f]; break;
                case STAGE_AB2: {
                    const double2 h = a.H[o];
                    a.S[o] = make_double2(S[f].x + dt * (1.5 * R[f].x - 0.5 * h.x), S[f].y + dt * (1.5 * R[f].y - 0.5 * h.y));
                    a.H[o] = R[f];
                } break;
                case STAGE_RK4_1: a.H[o] = S[f]; a.Acc[o] = axpy(S[f], dt / 6.0, R[f]); a.S[o] = axpy(S[f], 0.5 * dt, R[f]); break;
                case STAGE_RK4_2: a.Acc[o] = axpy(a.Acc[o], dt / 3.0, R[f]); a.S[o] = axpy(a.H[o], 0.5 * dt, R[f]); break;
                case STAGE_RK4_3: a.Acc[o] = axpy(a.Acc[o], dt / 3.0, R[f]); a.S[o] = axpy(a.H[o], dt, R[f]); break;
                default: a.S[o] = axpy(a.Acc[o], dt / 6.0, R[f]); break;   // STAGE_RK4_4
            }
        }
    }
}

cudaError_t launch_stage(const StageArgs& a, cudaStream_t st) {
    long long blocks = (a.g.field + kThreads - 1) / kThreads;
    if (blocks > kGridStream) blocks = kGridStream;
    if (a.hydro) stage_kernel<1><<<(unsigned)blocks, kThreads, 0, st>>>(a);
    else if (MHD_STAGE_SPLIT) {
        stage_kernel<1><<<(unsigned)blocks, kThreads, 0, st>>>(a);
        count_launch();
        stage_kernel<2><<<(unsigned)blocks, kThreads, 0, st>>>(a);
    } else stage_kernel<0><<<(unsigned)blocks, kThreads, 0, st>>>(a);
    count_launch();
    return cudaGetLastError();
}

// ---- S5: diagnostics -----------------------------------------------------------------------------
__global__ void divb_spec_kernel(SpecGeom g, const double2* __restrict__ B, double2* __restrict__ out, double kfx, double kfy, double kfz) {
    const long long F = g.field;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < F; idx += (long long)gridDim.x * blockDim.x) {
        const int jx = (int)(idx % g.px);
        const long long row = idx / g.px;
        const int jy = (int)(row % g.nky), jz = (int)(row / g.nky);
        double2 r = make_double2(0.0, 0.0);
        if (jx < g.nkx) {
            const double kx = kfx * (double)jx, ky = kfy * wavenum(jy, g.nky), kz = kfz * wavenum(jz, g.nkz);
            const double2 bx = B[idx], by = B[F + idx], bz = B[2 * F + idx];
            const double dx = kx * bx.x + ky * by.x + kz * bz.x, dy = kx * bx.y + ky * by.y + kz * bz.y;
            r = make_double2(-dy, dx);   // i * (k.B^)
        }
        out[idx] = r;
    }
}
cudaError_t launch_divb_spec(const SpecGeom& g, const double2* B, double2* out, double kfx, double kfy, double kfz, cudaStream_t st) {
    long long blocks = (g.field + kThreads - 1) / kThreads;
    if (blocks > kGridStream) blocks = kGridStream;
    divb_spec_kernel<<<(unsigned)blocks, kThreads, 0, st>>>(g, B, out, kfx, kfy, kfz);
    count_launch();
    return cudaGetLastError();
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// block-wide sum of NV values per thread; result valid in thread 0.  Fixed tree => deterministic.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* sm /* [NV][warps] */) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
        const double s = warp_sum(v[j]);
        if (lane == 0) sm[j * nw + w] = s;
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            double s = (lane < nw) ? sm[j * nw + lane] : 0.0;
            v[j] = warp_sum(s);
        }
    }
    __syncthreads();
}

template <bool HYDRO>
__global__ void __launch_bounds__(kThreads) reduce_fields_kernel(const double* __restrict__ f, long long npts, double* __restrict__ partial) {
    __shared__ double sm[(RED_NSUM + 1) * (kThreads / 32)];
    double v[RED_NSUM + 1];
#pragma unroll
    for (int j = 0; j <= RED_NSUM; ++j) v[j] = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < npts; i += (long long)gridDim.x * blockDim.x) {
        const double r = f[F_RHO * npts + i], mx = f[F_MX * npts + i], my = f[F_MY * npts + i], mz = f[F_MZ * npts + i];
        double bx = 0.0, by = 0.0, bz = 0.0;
        if (!HYDRO) { bx = f[F_BX * npts + i]; by = f[F_BY * npts + i]; bz = f[F_BZ * npts + i]; }
        v[0] += 0.5 * (mx * mx + my * my + mz * mz) / r;
        v[1] += 0.5 * (bx * bx + by * by + bz * bz);
        v[2] += r * log(r);
        v[3] += r; v[4] += mx; v[5] += my; v[6] += mz; v[7] += bx; v[8] += by; v[9] += bz;
        const bool fin = isfinite(r) && isfinite(mx) && isfinite(my) && isfinite(mz) && isfinite(bx) && isfinite(by) && isfinite(bz);
        if (!(r > 0.0) || !fin) v[RED_NSUM] = 1.0;
    }
    block_sum<RED_NSUM + 1>(v, sm);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int j = 0; j <= RED_NSUM; ++j) partial[(long long)j * gridDim.x + blockIdx.x] = v[j];
    }
}

// one block: results[j] = sum_b partial[j][b]
__global__ void __launch_bounds__(kThreads) reduce_final_sum_kernel(const double* __restrict__ partial, int nblocks, int nv, double* __restrict__ results) {
    __shared__ double sm[kThreads / 32];
    for (int j = 0; j < nv; ++j) {
        double v[1] = {0.0};
        for (int b = threadIdx.x; b < nblocks; b += blockDim.x) v[0] += partial[(long long)j * nblocks + b];
        block_sum<1>(v, sm);
        if (threadIdx.x == 0) results[j] = v[0];
    }
}

cudaError_t launch_reduce_fields(const double* f, long long npts, int hydro, double* partial, double* results, cudaStream_t st) {
    if (hydro) reduce_fields_kernel<true><<<RED_BLOCKS, kThreads, 0, st>>>(f, npts, partial);
    else reduce_fields_kernel<false><<<RED_BLOCKS, kThreads, 0, st>>>(f, npts, partial);
    count_launch();
    reduce_final_sum_kernel<<<1, kThreads, 0, st>>>(partial, RED_BLOCKS, RED_NSUM + 1, results);
    count_launch();
    return cudaGetLastError();
}

__global__ void __launch_bounds__(kThreads) reduce_maxabs_kernel(const double* __restrict__ a, long long npts, double* __restrict__ partial) {
    __shared__ double sm[2 * (kThreads / 32)];
    double mx = 0.0, bad = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < npts; i += (long long)gridDim.x * blockDim.x) {
        const double v = fabs(a[i]);
        mx = fmax(mx, v);
        if (!isfinite(v)) bad = 1.0;
    }
    mx = warp_max(mx); bad = warp_max(bad);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (lane == 0) { sm[w] = mx; sm[nw + w] = bad; }
    __syncthreads();
    if (w == 0) {
        mx = warp_max(lane < nw ? sm[lane] : 0.0);
        bad = warp_max(lane < nw ? sm[nw + lane] : 0.0);
        if (lane == 0) { partial[blockIdx.x] = mx; partial[gridDim.x + blockIdx.x] = bad; }
    }
}
__global__ void __launch_bounds__(kThreads) reduce_final_max_kernel(const double* __restrict__ partial, int nblocks, double* __restrict__ result) {
    __shared__ double sm[2 * (kThreads / 32)];
    double mx = 0.0, bad = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) { mx = fmax(mx, partial[b]); bad = fmax(bad, partial[nblocks + b]); }
    mx = warp_max(mx); bad = warp_max(bad);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (lane == 0) { sm[w] = mx; sm[nw + w] = bad; }
    __syncthreads();
    if (w == 0) {
        mx = warp_max(lane < nw ? sm[lane] : 0.0);
        bad = warp_max(lane < nw ? sm[nw + lane] : 0.0);
        if (lane == 0) { result[0] = mx; result[1] = bad; }
    }
}
cudaError_t launch_reduce_maxabs(const double* a, long long npts, double* partial, double* result, cudaStream_t st) {
    reduce_maxabs_kernel<<<RED_BLOCKS, kThreads, 0, st>>>(a, npts, partial);
    count_launch();
    reduce_final_max_kernel<<<1, kThreads, 0, st>>>(partial, RED_BLOCKS, result);
    count_launch();
    return cudaGetLastError();
}

// ---- paper diagnostics: sum_k w |k x V^|^2 and sum_k w |V^|^2 over a 3-component spectrum (Parseval) ---------
// Omega(t) = <|curl u|^2> and the terms of the Rayleigh quotient eq. (14).
// Half-spectrum entries with 0 < kx < nx/2 stand for two modes (w = 2).  Fixed grid + fixed tree: deterministic.
__global__ void __launch_bounds__(kThreads) reduce_curl_kernel(SpecGeom g, const double2* __restrict__ V, double kfx, double kfy, double kfz,
                                                               double* __restrict__ partial) {
    __shared__ double sm[2 * (kThreads / 32)];
    const long long F = g.field;
    double v[2] = {0.0, 0.0};
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < F; idx += (long long)gridDim.x * blockDim.x) {
        const int jx = (int)(idx % g.px);
        if (jx >= g.nkx) continue;
        const long long row = idx / g.px;
        const int jy = (int)(row % g.nky), jz = (int)(row / g.nky);
        const double kx = kfx * (double)jx, ky = kfy * wavenum(jy, g.nky), kz = kfz * wavenum(jz, g.nkz);
        const double w = (jx == 0 || 2 * jx == g.nx) ? 1.0 : 2.0;
        const double2 a = V[idx], b = V[F + idx], c = V[2 * F + idx];
        const double wxr = ky * c.x - kz * b.x, wxi = ky * c.y - kz * b.y;
        const double wyr = kz * a.x - kx * c.x, wyi = kz * a.y - kx * c.y;
        const double wzr = kx * b.x - ky * a.x, wzi = kx * b.y - ky * a.y;
        v[0] += w * (wxr * wxr + wxi * wxi + wyr * wyr + wyi * wyi + wzr * wzr + wzi * wzi);
        v[1] += w * (a.x * a.x + a.y * a.y + b.x * b.x + b.y * b.y + c.x * c.x + c.y * c.y);
    }
    block_sum<2>(v, sm);
    if (threadIdx.x == 0) { partial[blockIdx.x] = v[0]; partial[gridDim.x + blockIdx.x] = v[1]; }
}
cudaError_t launch_reduce_curl(const SpecGeom& g, const double2* V3, double kfx, double kfy, double kfz, double* partial, double* results,
                               cudaStream_t st) {
    reduce_curl_kernel<<<RED_BLOCKS, kThreads, 0, st>>>(g, V3, kfx, kfy, kfz, partial);
    count_launch();
    reduce_final_sum_kernel<<<1, kThreads, 0, st>>>(partial, RED_BLOCKS, 2, results);
    count_launch();
    return cudaGetLastError();
}

// ---- shell spectra, deterministic ------------------------------------------------------------------
// Along a row (fixed ky, kz) the shell index s = round(|k|) is non-decreasing in kx and grows by at
// most 1 per step, so one thread per row writes run sums into rowbins[row][s - s0(row)]; then one
// block per shell gathers over the rows in a fixed order.
__device__ __forceinline__ int shell_of(double k2) { return (int)floor(sqrt(k2) + 0.5); }

__global__ void __launch_bounds__(kThreads) spectra_rows_kernel(SpecGeom g, const double2* __restrict__ V, double* __restrict__ bins) {
    const long long rows = (long long)g.nky * g.nkz;
    const long long row = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= rows) return;
    const int jy = (int)(row % g.nky), jz = (int)(row / g.nky);
    const double ky = wavenum(jy, g.nky), kz = wavenum(jz, g.nkz);
    const double kyz2 = ky * ky + kz * kz;
    const int s0 = shell_of(kyz2);
    const long long F = g.field, base = row * g.px;
    double* __restrict__ bk = bins + row * g.nkx;
    int cur = s0;
    double acc = 0.0;
    for (int jx = 0; jx < g.nkx; ++jx) {
        const int s = shell_of(kyz2 + (double)jx * (double)jx);
        if (s != cur) {
            bk[cur - s0] = acc;
            for (int t = cur + 1; t < s; ++t) bk[t - s0] = 0.0;
            cur = s; acc = 0.0;
        }
        const double w = (jx == 0 || 2 * jx == g.nx) ? 0.5 : 1.0;   // 1/2 * (1 or 2 modes)
        double pw = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double2 v = V[c * F + base + jx];
            pw += v.x * v.x + v.y * v.y;
        }
        acc += w * pw;
    }
    bk[cur - s0] = acc;
    for (int t = cur - s0 + 1; t < g.nkx; ++t) bk[t] = 0.0;
}

__global__ void __launch_bounds__(kThreads) spectra_gather_kernel(SpecGeom g, const double* __restrict__ bins, double* __restrict__ spec, double norm) {
    __shared__ double sm[kThreads / 32];
    const int s = blockIdx.x;
    const long long rows = (long long)g.nky * g.nkz;
    double v[1] = {0.0};
    for (long long row = threadIdx.x; row < rows; row += blockDim.x) {
        const int jy = (int)(row % g.nky), jz = (int)(row / g.nky);
        const double ky = wavenum(jy, g.nky), kz = wavenum(jz, g.nkz);
        const int d = s - shell_of(ky * ky + kz * kz);
        if (d >= 0 && d < g.nkx) v[0] += bins[row * g.nkx + d];
    }
    block_sum<1>(v, sm);
    if (threadIdx.x == 0) spec[s] = v[0] * norm;
}

// shell spectrum of one 3-component spectral field V3 stored in geometry g; rowbins: rows*nkx doubles of scratch
cudaError_t launch_spectrum(const SpecGeom& g, const double2* V3, double* rowbins, double* spec, int nshell, cudaStream_t st) {
    const long long rows = (long long)g.nky * g.nkz;
    const unsigned blocks = (unsigned)((rows + kThreads - 1) / kThreads);
    spectra_rows_kernel<<<blocks, kThreads, 0, st>>>(g, V3, rowbins);
    count_launch();
    const double npts = (double)g.nx * (double)g.ny * (double)g.nz;
    spectra_gather_kernel<<<nshell, kThreads, 0, st>>>(g, rowbins, spec, 1.0 / (npts * npts));
    count_launch();
    return cudaGetLastError();
}

}  // namespace mhd
