// planefft_kernel.cu — the x and y passes of a batched 3-D real FFT in ONE persistent kernel, plane by plane through L2
// (the "2-sweep" transform of SURVEY.md §8(d) / §8(f) #4 for mhd_fft_r2c / mhd_fft_c2r, BASELINE config 5).
//
// The FFT under the pseudo-spectral derivative (the paper calls cuFFT/AccFFT) is three
// 1-D passes.  Run as three kernels, every pass streams the whole batch through HBM (6 F per transform).  Here the x and
// y passes of an (x,y) plane meet in a small ring of plane groups that lives in L2 (a 512 x 257 complex plane is 2.1 MB;
// the ring holds a few of them, against 126 MB of L2): the x pass of group g+LAG and the y pass of group g are in flight
// together, the intermediate never needs HBM, and the transform moves 4 F.
//
//   R2C:  phase A = x rows   (real rows -> half-spectrum rows into the ring),   phase B = y columns (ring -> out)
//   C2R:  phase A = y columns (in -> ring),                                     phase B = x rows   (ring -> real rows)
//
// Scheduling: work items are handed out IN ORDER by one global counter:  A(0) .. A(LAG-1), then A(t) B(t-LAG) for
// t = LAG .., then the remaining B.  A B item waits (acquire spin on a per-group counter) until all A items of its
// group have signalled (release); an A item of group g waits for all B items of group g-RING, whose slot it overwrites.
// Dependencies only point backwards in the hand-out order, so the oldest unfinished item can always run: no deadlock,
// whatever the number of resident CTAs.  In steady state nothing waits: a producer is LAG groups ahead of its consumer.
// Ring data is moved with ld.global.cg / st.global.cg (L2 only: no stale L1 lines when a slot is reused).
//
// x rows use the team machinery of xteam.cuh (coalesced rows, two real rows per complex transform); y columns use the
// 8-column tiles of fft_core.cuh (one 128-byte line per row).  512 threads per CTA, <= 64 registers, ~82 KB of shared
// memory: two CTAs per SM.
#include "mhd_internal.h"
#include "xteam.cuh"

namespace mhd {
using namespace mhdfft;

template <int N> struct PlaneCfg {
    static constexpr int THREADS = 512;
    static constexpr int TP = Plan<N>::TP;
    static constexpr int TEAMS = THREADS / TP;                   // row pairs per x item
    static constexpr int COLG = THREADS / (8 * TP);              // 8-column groups per y item
    static constexpr int COLS = 8 * COLG;
    static constexpr int BUF = Padded::size(N);
    static constexpr int NTW = XCfg<N>::NTW > 0 ? XCfg<N>::NTW : 1;
    static constexpr size_t XS = sizeof(cplx) * (size_t)BUF * TEAMS;
    static constexpr size_t YS = sizeof(cplx) * (size_t)N * COLS;
    static constexpr size_t SMEM = (XS > YS ? XS : YS) + sizeof(cplx) * NTW;
    static_assert(Plan<N>::E == 8 && THREADS % (8 * TP) == 0, "plane kernel: lengths 64..512 with 8 points per thread");
};

__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// all threads of the CTA: wait until *flag >= need
__device__ __forceinline__ void cta_wait(const unsigned* flag, unsigned need) {
    if (threadIdx.x == 0) {
        while (ld_acquire(flag) < need) __nanosleep(64);
    }
    __syncthreads();
}
// all threads of the CTA have issued their global writes: publish them and count the item
__device__ __forceinline__ void cta_signal(unsigned* flag) {
    __syncthreads();
    if (threadIdx.x == 0) red_release(flag, 1u);
}

template <int N, bool INV>
__global__ void __launch_bounds__(PlaneCfg<N>::THREADS, 2) planefft_kernel(PlaneFftArgs a, const cplx* __restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smraw[];
    using PL = Plan<N>;
    using PC = PlaneCfg<N>;
    constexpr int TP = PL::TP, E = 8, RL = PL::radix(PL::NP - 1);
    cplx* const smbase = reinterpret_cast<cplx*>(smraw);
    cplx* const stw = reinterpret_cast<cplx*>(smraw + (PC::XS > PC::YS ? PC::XS : PC::YS));
    __shared__ long long s_item;

    // per-pass twiddle tables for the team passes
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

    const int nxh = a.nxh, pitch = a.pitch, G = a.group;
    const long long plane_ring = (long long)N * pitch;                  // complex per plane in the ring
    // items per group: x rows and y column tiles (planes past the end of the batch are skipped but still counted)
    const int nX = G * ((N / 2 + PC::TEAMS - 1) / PC::TEAMS);
    const int ytiles = (nxh + PC::COLS - 1) / PC::COLS;
    const int nY = G * ytiles;
    const int nA = INV ? nY : nX, nB = INV ? nX : nY;
    const long long NG = a.ngroups, LAG = a.lag;
    const long long head = LAG < NG ? LAG : NG;                          // groups whose A phase runs before any B phase
    const long long total = NG * (long long)(nA + nB);
    unsigned* const doneA = a.counters + 4;
    unsigned* const doneB = doneA + NG;

    // ---- x rows of one item: row pairs (team) of plane `pl` of group g ----
    auto x_item = [&](long long g, int idx) {
        const int team = threadIdx.x / TP, i = threadIdx.x % TP;
        cplx* const buf = smbase + (size_t)team * PC::BUF;
        const int per_plane = (N / 2 + PC::TEAMS - 1) / PC::TEAMS;
        const int pl = idx / per_plane, blk = idx % per_plane;
        const long long plane = g * G + pl;
        const int pr = blk * PC::TEAMS + team;                            // row pair within the plane
        const bool ok = plane < a.nplanes && pr < N / 2;
        const cplx* __restrict__ ringc = a.ring + ((g % a.ring_slots) * G + pl) * plane_ring + (long long)(2 * pr) * pitch;
        cplx* __restrict__ ring = const_cast<cplx*>(ringc);
        double* __restrict__ ra = a.real + ((ok ? plane : 0) * N + (ok ? 2 * pr : 0)) * (long long)N;
        double* __restrict__ rb = ra + N;
        cplx v[E];
        if constexpr (INV) {
#pragma unroll
            for (int q = 0; q < E; ++q) {                 // first-pass input k = i + TP*q
                const int k = i + TP * q;
                const bool lo = k < nxh, hi = (N - k) < nxh;
                const int idxk = lo ? k : N - k;
                cplx x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
                if (ok && (lo || hi)) { x = __ldcg(&ringc[idxk]); y = __ldcg(&ringc[pitch + idxk]); }
                if (k == 0 || 2 * k == N) { x.y = 0.0; y.y = 0.0; }                 // self-conjugate modes: Im ignored
                v[q] = lo ? make_double2(x.x - y.y, x.y + y.x) : make_double2(x.x + y.y, y.x - x.y);
            }
            XPass<N, true, 0, 1, true>::run(v, buf, buf, i, team, stw);
            const double s = a.scale;
            if (ok) {
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int x = i + TP * (m + q * (E / RL));
                        __stcs(&ra[x], v[m * RL + q].x * s);
                        __stcs(&rb[x], v[m * RL + q].y * s);
                    }
            }
        } else {
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = ok ? make_double2(__ldcs(&ra[i + TP * q]), __ldcs(&rb[i + TP * q])) : make_double2(0.0, 0.0);
            XPass<N, false, 0, 1, true>::run(v, buf, buf, i, team, stw);
            // Hermitian split: A[k] = (Z[k] + conj Z[N-k])/2, B[k] = (Z[k] - conj Z[N-k])/(2i); only Z[N-k] crosses threads
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int t = m + q * (E / RL);
                    if (t >= 1 && (TP * (t + 1) > N - nxh)) buf[N - (i + TP * t)] = v[m * RL + q];
                }
            team_sync<TP>(team);
            if (ok) {
#pragma unroll
                for (int m = 0; m < E / RL; ++m)
#pragma unroll
                    for (int q = 0; q < RL; ++q) {
                        const int t = m + q * (E / RL);
                        const int k = i + TP * t;
                        if (t <= E / 2 && k < nxh) {
                            const cplx zk = v[m * RL + q];
                            const cplx zm = (k == 0) ? zk : buf[k];
                            __stcg(&ring[k], make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y)));
                            __stcg(&ring[pitch + k], make_double2(0.5 * (zk.y + zm.y), 0.5 * (zm.x - zk.x)));
                        }
                    }
            }
            team_sync<TP>(team);          // the split reads of buf are done before the next item's first pass writes it
        }
    };

    // ---- y columns of one item: an 8*COLG-column tile of plane `pl` of group g ----
    auto y_item = [&](long long g, int idx) {
        const int tid = threadIdx.x, p = tid & 7, i = (tid >> 3) % TP, cg = tid / (8 * TP);
        cplx* const sm = smbase + (size_t)cg * N * 8;
        const int pl = idx / ytiles, tile = idx % ytiles;
        const long long plane = g * G + pl;
        const int col = tile * PC::COLS + cg * 8 + p;
        const bool ok = plane < a.nplanes && col < nxh;
        const cplx* __restrict__ ringc = a.ring + ((g % a.ring_slots) * G + pl) * plane_ring + col;
        cplx* __restrict__ ring = const_cast<cplx*>(ringc);
        const cplx* __restrict__ src = a.spec_in + (ok ? plane : 0) * (long long)N * nxh + col;      // INV: y columns of the input planes
        cplx* __restrict__ dst = a.spec_out + (ok ? plane : 0) * (long long)N * nxh + col;           // !INV: y columns of the output planes
        cplx v[E];
        constexpr int R0 = PL::radix(0);
#pragma unroll
        for (int m = 0; m < E / R0; ++m)
#pragma unroll
            for (int q = 0; q < R0; ++q) {
                const int r = first_index<N>(i, m, q);
                cplx x = make_double2(0.0, 0.0);
                if (ok) x = INV ? __ldcs(&src[(long long)r * nxh]) : __ldcg(&ringc[(long long)r * pitch]);
                v[m * R0 + q] = x;
            }
        pencil_fft<N, INV>(v, sm, i, p, tw);
        if (ok) {
#pragma unroll
            for (int m = 0; m < E / RL; ++m)
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const int r = last_index<N>(i, m, q);
                    if constexpr (INV) __stcg(&ring[(long long)r * pitch], v[m * RL + q]);
                    else __stcs(&dst[(long long)r * nxh], v[m * RL + q]);
                }
        }
        __syncthreads();                  // the exchange buffer is reused by the next item (x or y)
    };

    for (;;) {
        if (threadIdx.x == 0) s_item = (long long)atomicAdd(reinterpret_cast<unsigned long long*>(a.counters), 1ull);
        __syncthreads();
        const long long item = s_item;
        __syncthreads();
        if (item >= total) break;
        // decode: which phase of which group
        bool isA;
        long long g;
        int idx;
        const long long head_items = head * nA;
        const long long steady_items = (NG - head) * (long long)(nA + nB);
        if (item < head_items) {
            isA = true; g = item / nA; idx = (int)(item % nA);
        } else if (item < head_items + steady_items) {
            const long long r = item - head_items;
            const long long t = head + r / (nA + nB);
            const int w = (int)(r % (nA + nB));
            if (w < nA) { isA = true; g = t; idx = w; }
            else { isA = false; g = t - head; idx = w - nA; }
        } else {
            const long long r = item - head_items - steady_items;
            isA = false; g = (NG - head) + r / nB; idx = (int)(r % nB);
        }
        if (isA) {
            if (g >= a.ring_slots) cta_wait(&doneB[g - a.ring_slots], (unsigned)nB);     // the slot's previous tenant has been consumed
            if constexpr (INV) y_item(g, idx); else x_item(g, idx);
            cta_signal(&doneA[g]);
        } else {
            cta_wait(&doneA[g], (unsigned)nA);
            if constexpr (INV) x_item(g, idx); else y_item(g, idx);
            cta_signal(&doneB[g]);
        }
    }
}

size_t planefft_counter_bytes(long long nplanes, int group) {
    const long long ng = (nplanes + group - 1) / group;
    return sizeof(unsigned) * (size_t)(4 + 2 * ng);
}

bool planefft_supported(int nx, int ny) {
    if (nx != ny) return false;
    return nx == 64 || nx == 128 || nx == 256 || nx == 512;
}

template <int N> static cudaError_t launch_planefft_n(bool inverse, const PlaneFftArgs& a, const cplx* tw, cudaStream_t st) {
    using PC = PlaneCfg<N>;
    static DeviceOnce once;
    const int dev = device_slot();
    if (dev < 0) return cudaErrorInvalidDevice;
    int sms = 0;
    cudaError_t e = device_sm_count(dev, &sms);
    if (e != cudaSuccess) return e;
    if (!once.done[dev]) {
        e = cudaFuncSetAttribute(planefft_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PC::SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(planefft_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PC::SMEM);
        if (e != cudaSuccess) return e;
        once.done[dev] = true;
    }
    e = cudaMemsetAsync(a.counters, 0, planefft_counter_bytes(a.nplanes, a.group), st);
    if (e != cudaSuccess) return e;
    const unsigned blocks = (unsigned)(sms * 2);
    if (inverse) planefft_kernel<N, true><<<blocks, PC::THREADS, PC::SMEM, st>>>(a, tw);
    else planefft_kernel<N, false><<<blocks, PC::THREADS, PC::SMEM, st>>>(a, tw);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_planefft(int n, bool inverse, const PlaneFftArgs& a, const double2* tw, cudaStream_t st) {
    switch (n) {
        case 64: return launch_planefft_n<64>(inverse, a, tw, st);
        case 128: return launch_planefft_n<128>(inverse, a, tw, st);
        case 256: return launch_planefft_n<256>(inverse, a, tw, st);
        case 512: return launch_planefft_n<512>(inverse, a, tw, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace mhd
