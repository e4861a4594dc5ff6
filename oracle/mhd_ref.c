/* mhd_ref.c — CPU ORACLE (test infrastructure only; see mhd_ref.h for scope, citations and pins).
 *
 * Plain C99, fp64, no blocking / fusion / reordering beyond what the algorithm states.
 * OpenMP is used only on loops whose iterations are independent (rows, pencils, points), so the
 * result does not depend on the thread count.  Reductions are serial and compensated.
 */
#include "mhd_ref.h"

#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

static int g_threads = 0; /* 0 = OpenMP default */

void mhd_ref_set_threads(int n) {
    g_threads = n > 0 ? n : 0;
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#endif
}
int mhd_ref_get_threads(void) {
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * 1-D FFT: recursive decimation in time over the smallest prime factor; a prime length falls
 * through to the O(n^2) definition.  X[k] = sum_j x[j] w^(jk), w = exp(sign*2*pi*i/n).
 * tw[j] = exp(sign*2*pi*i*j/N) for the top-level length N (computed in long double).
 * ------------------------------------------------------------------------------------------ */
static int smallest_factor(int n) {
    for (int p = 2; p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

static void fft_rec(int n, int N, const cplx* tw, const cplx* in, int istride, cplx* out) {
    if (n == 1) { out[0] = in[0]; return; }
    int r = smallest_factor(n), m = n / r, step = N / n;
    /* r sub-transforms of length m over the decimated sequences x[q], x[q+r], x[q+2r], ... */
    for (int q = 0; q < r; ++q) fft_rec(m, N, tw, in + (size_t)q * istride, istride * r, out + (size_t)q * m);
    /* combine: X[k + p*m] = sum_q w_n^(q*(k+p*m)) * Y_q[k] */
    cplx y[64], *yy = y;
    if (r > 64) yy = (cplx*)malloc(sizeof(cplx) * (size_t)r);
    for (int k = 0; k < m; ++k) {
        for (int q = 0; q < r; ++q) yy[q] = out[(size_t)q * m + k];
        for (int p = 0; p < r; ++p) {
            int kk = k + p * m;
            cplx acc = 0.0;
            for (int q = 0; q < r; ++q) acc += tw[(size_t)(((long long)q * kk) % n) * step] * yy[q];
            out[(size_t)p * m + k] = acc;
        }
    }
    if (yy != y) free(yy);
}

typedef struct { int n; cplx* fwd; cplx* inv; } twiddles;

static int tw_init(twiddles* t, int n) {
    t->n = n;
    t->fwd = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    t->inv = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    if (!t->fwd || !t->inv) return -1;
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int j = 0; j < n; ++j) {
        long double a = two_pi * (long double)j / (long double)n;
        double c = (double)cosl(a), s = (double)sinl(a);
        t->fwd[j] = c - I * s;
        t->inv[j] = c + I * s;
    }
    return 0;
}
static void tw_free(twiddles* t) { free(t->fwd); free(t->inv); t->fwd = t->inv = NULL; }

int mhd_ref_fft1d(int n, int sign, const double* in, double* out) {
    if (n < 1 || !in || !out || (sign != 1 && sign != -1)) return MHD_REF_EINVAL;
    twiddles t;
    if (tw_init(&t, n)) return MHD_REF_ENOMEM;
    cplx* tmp = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    fft_rec(n, n, sign < 0 ? t.fwd : t.inv, (const cplx*)in, 1, tmp);
    memcpy(out, tmp, sizeof(cplx) * (size_t)n);
    free(tmp);
    tw_free(&t);
    return MHD_REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * 3-D transforms of one field.  R2C: x (real row -> full complex row, keep kx <= nx/2), then y,
 * then z.  C2R: z, then y, then x: rebuild the full Hermitian row X[nx-k] = conj(X[k]),
 * inverse-transform it, take the real part, divide by nx*ny*nz.
 * ------------------------------------------------------------------------------------------ */
typedef struct { int nx, ny, nz, nxh; twiddles tx, ty, tz; } plan3;

static int plan3_init(plan3* p, int nx, int ny, int nz) {
    p->nx = nx; p->ny = ny; p->nz = nz; p->nxh = nx / 2 + 1;
    if (tw_init(&p->tx, nx) || tw_init(&p->ty, ny) || tw_init(&p->tz, nz)) return -1;
    return 0;
}
static void plan3_free(plan3* p) { tw_free(&p->tx); tw_free(&p->ty); tw_free(&p->tz); }

/* in-place transform along a strided axis of a half-spectrum array */
static void axis_pass(cplx* a, int n, size_t stride, size_t npencil, const cplx* tw,
                      size_t outer_stride, size_t inner_count) {
    /* pencil p -> base offset (p / inner_count) * outer_stride + (p % inner_count) */
#pragma omp parallel
    {
        cplx* buf = (cplx*)malloc(sizeof(cplx) * 2 * (size_t)n);
        cplx* res = buf + n;
#pragma omp for schedule(static)
        for (long long p = 0; p < (long long)npencil; ++p) {
            size_t base = ((size_t)p / inner_count) * outer_stride + ((size_t)p % inner_count);
            for (int j = 0; j < n; ++j) buf[j] = a[base + (size_t)j * stride];
            fft_rec(n, n, tw, buf, 1, res);
            for (int j = 0; j < n; ++j) a[base + (size_t)j * stride] = res[j];
        }
        free(buf);
    }
}

static void r2c3(const plan3* p, const double* in, cplx* out) {
    const int nx = p->nx, ny = p->ny, nz = p->nz, nxh = p->nxh;
    const size_t rows = (size_t)ny * nz;
#pragma omp parallel
    {
        cplx* buf = (cplx*)malloc(sizeof(cplx) * 2 * (size_t)nx);
        cplx* res = buf + nx;
#pragma omp for schedule(static)
        for (long long r = 0; r < (long long)rows; ++r) {
            for (int j = 0; j < nx; ++j) buf[j] = in[(size_t)r * nx + j];
            fft_rec(nx, nx, p->tx.fwd, buf, 1, res);
            for (int k = 0; k < nxh; ++k) out[(size_t)r * nxh + k] = res[k];
        }
        free(buf);
    }
    /* y: for every (z, kx) */
    axis_pass(out, ny, (size_t)nxh, (size_t)nz * nxh, p->ty.fwd, (size_t)ny * nxh, (size_t)nxh);
    /* z: for every (ky, kx) */
    axis_pass(out, nz, (size_t)ny * nxh, (size_t)ny * nxh, p->tz.fwd, 0, (size_t)ny * nxh);
}

/* destroys `in` (used as work space) */
static void c2r3(const plan3* p, cplx* in, double* out) {
    const int nx = p->nx, ny = p->ny, nz = p->nz, nxh = p->nxh;
    const size_t rows = (size_t)ny * nz;
    const double scale = 1.0 / ((double)nx * (double)ny * (double)nz);
    axis_pass(in, nz, (size_t)ny * nxh, (size_t)ny * nxh, p->tz.inv, 0, (size_t)ny * nxh);
    axis_pass(in, ny, (size_t)nxh, (size_t)nz * nxh, p->ty.inv, (size_t)ny * nxh, (size_t)nxh);
#pragma omp parallel
    {
        cplx* buf = (cplx*)malloc(sizeof(cplx) * 2 * (size_t)nx);
        cplx* res = buf + nx;
#pragma omp for schedule(static)
        for (long long r = 0; r < (long long)rows; ++r) {
            for (int k = 0; k < nxh; ++k) buf[k] = in[(size_t)r * nxh + k];
            for (int k = nxh; k < nx; ++k) buf[k] = conj(in[(size_t)r * nxh + (nx - k)]);
            fft_rec(nx, nx, p->tx.inv, buf, 1, res);
            for (int j = 0; j < nx; ++j) out[(size_t)r * nx + j] = creal(res[j]) * scale;
        }
        free(buf);
    }
}

int mhd_ref_fft_r2c(int nx, int ny, int nz, int batch, const double* in, double* out) {
    if (nx < 1 || ny < 1 || nz < 1 || batch < 1 || !in || !out) return MHD_REF_EINVAL;
    plan3 p;
    if (plan3_init(&p, nx, ny, nz)) return MHD_REF_ENOMEM;
    size_t nr = (size_t)nx * ny * nz, nc = (size_t)p.nxh * ny * nz;
    for (int b = 0; b < batch; ++b) r2c3(&p, in + (size_t)b * nr, (cplx*)out + (size_t)b * nc);
    plan3_free(&p);
    return MHD_REF_OK;
}

int mhd_ref_fft_c2r(int nx, int ny, int nz, int batch, const double* in, double* out) {
    if (nx < 1 || ny < 1 || nz < 1 || batch < 1 || !in || !out) return MHD_REF_EINVAL;
    plan3 p;
    if (plan3_init(&p, nx, ny, nz)) return MHD_REF_ENOMEM;
    size_t nr = (size_t)nx * ny * nz, nc = (size_t)p.nxh * ny * nz;
    cplx* tmp = (cplx*)malloc(sizeof(cplx) * nc);
    if (!tmp) { plan3_free(&p); return MHD_REF_ENOMEM; }
    for (int b = 0; b < batch; ++b) {
        memcpy(tmp, (const cplx*)in + (size_t)b * nc, sizeof(cplx) * nc);
        c2r3(&p, tmp, out + (size_t)b * nr);
    }
    free(tmp);
    plan3_free(&p);
    return MHD_REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * Solver context
 * ------------------------------------------------------------------------------------------ */
enum { F_RHO = 0, F_MX, F_MY, F_MZ, F_BX, F_BY, F_BZ, NFIELD };
/* the 12 real-space products of SURVEY.md §8(a) S2 */
enum { P_TXX = 0, P_TYY, P_TZZ, P_TXY, P_TXZ, P_TYZ, P_EX, P_EY, P_EZ, P_UX, P_UY, P_UZ, NPROD };

struct mhd_ref_ctx {
    int nx, ny, nz, nxh;
    double nu, eta, cs, dt;
    int integrator;
    unsigned flags;
    plan3 plan;
    size_t nr, nc;          /* points per real field, modes per half-spectrum */
    cplx* S[NFIELD];        /* spectral state  rho^, m^, B^            */
    cplx* R[NFIELD];        /* right-hand side of the current stage    */
    cplx* Rold[NFIELD];     /* AB2 history                              */
    cplx* S0[NFIELD];       /* RK4: state at the start of the step     */
    cplx* Acc[NFIELD];      /* RK4: weighted sum of stage slopes       */
    double* f[NFIELD];      /* real-space rho, m, B                    */
    double* g[NPROD];       /* real-space products                     */
    cplx* G[NPROD];         /* their transforms                        */
    cplx* tmp;              /* scratch half-spectrum (c2r3 destroys its input) */
    double kfac[3];         /* 2*pi/L_i: physical wavenumber = kfac[i] * integer index (1.0 on the 2*pi box) */
    cplx* Fh[3];            /* masked transform of the steady body force f of eq. (2), or NULL */
    int have_fields, have_history;
    long long step;
    double time;
};

/* integer wavenumber of FFT index j on an axis of length n: 0..ceil(n/2)-1, then negative */
static int wavenumber(int j, int n) { return (j < (n + 1) / 2) ? j : j - n; }

/* 2/3 rule, per axis: keep iff 3|k_i| < n_i */
static int mask_keep(const mhd_ref_ctx* c, int kx, int ky, int kz) {
    if (c->flags & MHD_REF_FLAG_NO_DEALIAS) return 1;
    return 3 * abs(kx) < c->nx && 3 * abs(ky) < c->ny && 3 * abs(kz) < c->nz;
}

static void free_ctx(mhd_ref_ctx* c) {
    if (!c) return;
    for (int i = 0; i < NFIELD; ++i) { free(c->S[i]); free(c->R[i]); free(c->Rold[i]); free(c->S0[i]); free(c->Acc[i]); free(c->f[i]); }
    for (int i = 0; i < NPROD; ++i) { free(c->g[i]); free(c->G[i]); }
    free(c->tmp);
    for (int i = 0; i < 3; ++i) free(c->Fh[i]);
    plan3_free(&c->plan);
    free(c);
}

int mhd_ref_create(mhd_ref_ctx** out, int nx, int ny, int nz, double nu, double eta, double cs, double dt,
                   int integrator, unsigned flags) {
    if (!out) return MHD_REF_EINVAL;
    *out = NULL;
    if (nx < 2 || ny < 1 || nz < 1 || (nx & 1)) return MHD_REF_EINVAL;
    if (!(nu >= 0.0) || !(eta >= 0.0) || !(cs >= 0.0) || !(dt > 0.0)) return MHD_REF_EINVAL;
    if (integrator != MHD_REF_AB2 && integrator != MHD_REF_RK4) return MHD_REF_EINVAL;
    mhd_ref_ctx* c = (mhd_ref_ctx*)calloc(1, sizeof(*c));
    if (!c) return MHD_REF_ENOMEM;
    c->nx = nx; c->ny = ny; c->nz = nz; c->nxh = nx / 2 + 1;
    c->nu = nu; c->eta = eta; c->cs = cs; c->dt = dt;
    c->integrator = integrator; c->flags = flags;
    c->nr = (size_t)nx * ny * nz; c->nc = (size_t)c->nxh * ny * nz;
    c->kfac[0] = c->kfac[1] = c->kfac[2] = 1.0;
    if (plan3_init(&c->plan, nx, ny, nz)) { free_ctx(c); return MHD_REF_ENOMEM; }
    int ok = 1;
    for (int i = 0; i < NFIELD; ++i) {
        ok &= (c->S[i] = (cplx*)calloc(c->nc, sizeof(cplx))) != NULL;
        ok &= (c->R[i] = (cplx*)calloc(c->nc, sizeof(cplx))) != NULL;
        if (integrator == MHD_REF_AB2) ok &= (c->Rold[i] = (cplx*)calloc(c->nc, sizeof(cplx))) != NULL;
        if (integrator == MHD_REF_RK4) {
            ok &= (c->S0[i] = (cplx*)calloc(c->nc, sizeof(cplx))) != NULL;
            ok &= (c->Acc[i] = (cplx*)calloc(c->nc, sizeof(cplx))) != NULL;
        }
        ok &= (c->f[i] = (double*)calloc(c->nr, sizeof(double))) != NULL;
    }
    for (int i = 0; i < NPROD; ++i) {
        ok &= (c->g[i] = (double*)calloc(c->nr, sizeof(double))) != NULL;
        ok &= (c->G[i] = (cplx*)calloc(c->nc, sizeof(cplx))) != NULL;
    }
    ok &= (c->tmp = (cplx*)calloc(c->nc, sizeof(cplx))) != NULL;
    if (!ok) { free_ctx(c); return MHD_REF_ENOMEM; }
    *out = c;
    return MHD_REF_OK;
}

void mhd_ref_destroy(mhd_ref_ctx* c) { free_ctx(c); }

int mhd_ref_mask(mhd_ref_ctx* c, unsigned char* out) {
    if (!c || !out) return MHD_REF_EINVAL;
    for (int jz = 0; jz < c->nz; ++jz)
        for (int jy = 0; jy < c->ny; ++jy)
            for (int jx = 0; jx < c->nxh; ++jx)
                out[((size_t)jz * c->ny + jy) * c->nxh + jx] =
                    (unsigned char)mask_keep(c, jx, wavenumber(jy, c->ny), wavenumber(jz, c->nz));
    return MHD_REF_OK;
}

/* multiply a half-spectrum by M(k) */
static void apply_mask(const mhd_ref_ctx* c, cplx* a) {
#pragma omp parallel for schedule(static)
    for (int jz = 0; jz < c->nz; ++jz)
        for (int jy = 0; jy < c->ny; ++jy)
            for (int jx = 0; jx < c->nxh; ++jx)
                if (!mask_keep(c, jx, wavenumber(jy, c->ny), wavenumber(jz, c->nz)))
                    a[((size_t)jz * c->ny + jy) * c->nxh + jx] = 0.0;
}

/* box lengths: k_i = (2*pi/L_i) n_i   (PAPER.md:161 uses Lx = 1, Ly = 2; every other test the 2*pi box) */
int mhd_ref_set_box(mhd_ref_ctx* c, double lx, double ly, double lz) {
    if (!c || !(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0) || !isfinite(lx) || !isfinite(ly) || !isfinite(lz)) return MHD_REF_EINVAL;
    const double two_pi = 6.283185307179586476925286766559;
    const double l[3] = {lx, ly, lz};
    for (int i = 0; i < 3; ++i) c->kfac[i] = (l[i] == two_pi) ? 1.0 : two_pi / l[i];
    return MHD_REF_OK;
}

/* steady body force f of eq. (2): stored as its masked transform */
int mhd_ref_set_forcing(mhd_ref_ctx* c, const double* fx, const double* fy, const double* fz) {
    if (!c) return MHD_REF_EINVAL;
    const double* f[3] = {fx, fy, fz};
    if (!fx && !fy && !fz) {
        for (int i = 0; i < 3; ++i) { free(c->Fh[i]); c->Fh[i] = NULL; }
        return MHD_REF_OK;
    }
    if (!fx || !fy || !fz) return MHD_REF_EINVAL;
    for (int i = 0; i < 3; ++i) {
        if (!c->Fh[i]) c->Fh[i] = (cplx*)calloc(c->nc, sizeof(cplx));
        if (!c->Fh[i]) return MHD_REF_ENOMEM;
        memcpy(c->g[0], f[i], sizeof(double) * c->nr);
        r2c3(&c->plan, c->g[0], c->Fh[i]);
        apply_mask(c, c->Fh[i]);
    }
    return MHD_REF_OK;
}

/* step 1 of SURVEY.md §8(c.2): m = rho*u; forward-FFT the 7 fields; mask; reset history */
int mhd_ref_set_fields(mhd_ref_ctx* c, const double* rho, const double* ux, const double* uy, const double* uz,
                       const double* bx, const double* by, const double* bz) {
    if (!c || !rho || !ux || !uy || !uz) return MHD_REF_EINVAL;
    const int hydro = (c->flags & MHD_REF_FLAG_HYDRO) != 0;
    if (!hydro && (!bx || !by || !bz)) return MHD_REF_EINVAL;
    const double* u[3] = {ux, uy, uz};
    const double* b[3] = {bx, by, bz};
    memcpy(c->f[F_RHO], rho, sizeof(double) * c->nr);
    for (int i = 0; i < 3; ++i) {
        double* m = c->f[F_MX + i];
#pragma omp parallel for schedule(static)
        for (long long p = 0; p < (long long)c->nr; ++p) m[p] = rho[p] * u[i][p];
        if (hydro) memset(c->f[F_BX + i], 0, sizeof(double) * c->nr);
        else memcpy(c->f[F_BX + i], b[i], sizeof(double) * c->nr);
    }
    for (int i = 0; i < NFIELD; ++i) {
        r2c3(&c->plan, c->f[i], c->S[i]);
        apply_mask(c, c->S[i]);
    }
    c->have_fields = 1; c->have_history = 0; c->step = 0; c->time = 0.0;
    return MHD_REF_OK;
}

/* inverse-transform the 7 spectral fields of `S` into c->f (real rho, m, B) */
static void to_real(mhd_ref_ctx* c, cplx* const* S) {
    for (int i = 0; i < NFIELD; ++i) {
        memcpy(c->tmp, S[i], sizeof(cplx) * c->nc);
        c2r3(&c->plan, c->tmp, c->f[i]);
    }
}

/* step 2 of SURVEY.md §8(c.2): R = RHS(S) */
static void rhs(mhd_ref_ctx* c, cplx* const* S, cplx* const* R) {
    const int hydro = (c->flags & MHD_REF_FLAG_HYDRO) != 0;
    const int nprod_first_skip = P_EX, nprod_last_skip = P_EZ; /* hydro: E = u x B is not needed */
    to_real(c, S);
    /* S2: real-space products (eq. 2: rho u u + (B^2/2) I - B B; eq. 4: u x B) */
    {
        const double *rho = c->f[F_RHO], *mx = c->f[F_MX], *my = c->f[F_MY], *mz = c->f[F_MZ];
        const double *bx = c->f[F_BX], *by = c->f[F_BY], *bz = c->f[F_BZ];
        double* const* g = c->g;
#pragma omp parallel for schedule(static)
        for (long long p = 0; p < (long long)c->nr; ++p) {
            double inv = 1.0 / rho[p];
            double ux = mx[p] * inv, uy = my[p] * inv, uz = mz[p] * inv;
            double Bx = hydro ? 0.0 : bx[p], By = hydro ? 0.0 : by[p], Bz = hydro ? 0.0 : bz[p];
            double b2h = 0.5 * (Bx * Bx + By * By + Bz * Bz);
            g[P_TXX][p] = mx[p] * ux + b2h - Bx * Bx;
            g[P_TYY][p] = my[p] * uy + b2h - By * By;
            g[P_TZZ][p] = mz[p] * uz + b2h - Bz * Bz;
            g[P_TXY][p] = mx[p] * uy - Bx * By;
            g[P_TXZ][p] = mx[p] * uz - Bx * Bz;
            g[P_TYZ][p] = my[p] * uz - By * Bz;
            g[P_EX][p] = uy * Bz - uz * By;
            g[P_EY][p] = uz * Bx - ux * Bz;
            g[P_EZ][p] = ux * By - uy * Bx;
            g[P_UX][p] = ux; g[P_UY][p] = uy; g[P_UZ][p] = uz;
        }
    }
    /* S3: forward transforms */
    for (int i = 0; i < NPROD; ++i) {
        if (hydro && i >= nprod_first_skip && i <= nprod_last_skip) continue;
        r2c3(&c->plan, c->g[i], c->G[i]);
    }
    /* S4: spectral assembly, mode by mode */
    const double nu = c->nu, eta = c->eta, cs2 = c->cs * c->cs;
    cplx* const* G = c->G;
#pragma omp parallel for schedule(static)
    for (int jz = 0; jz < c->nz; ++jz)
        for (int jy = 0; jy < c->ny; ++jy)
            for (int jx = 0; jx < c->nxh; ++jx) {
                size_t q = ((size_t)jz * c->ny + jy) * c->nxh + jx;
                int ny_ = wavenumber(jy, c->ny), nz_ = wavenumber(jz, c->nz);
                double kx = c->kfac[0] * jx, ky = c->kfac[1] * ny_, kz = c->kfac[2] * nz_;
                double k2 = kx * kx + ky * ky + kz * kz;
                double M = mask_keep(c, jx, ny_, nz_) ? 1.0 : 0.0;
                /* eq. (1): d rho/dt = -div m */
                R[F_RHO][q] = -I * (kx * S[F_MX][q] + ky * S[F_MY][q] + kz * S[F_MZ][q]);
                /* eq. (2)+(3): d m_i/dt = -d_j T_ij - cs^2 d_i rho + nu lap u_i */
                R[F_MX][q] = M * (-I * (kx * G[P_TXX][q] + ky * G[P_TXY][q] + kz * G[P_TXZ][q])
                                  - I * kx * cs2 * S[F_RHO][q] - nu * k2 * G[P_UX][q]);
                R[F_MY][q] = M * (-I * (kx * G[P_TXY][q] + ky * G[P_TYY][q] + kz * G[P_TYZ][q])
                                  - I * ky * cs2 * S[F_RHO][q] - nu * k2 * G[P_UY][q]);
                R[F_MZ][q] = M * (-I * (kx * G[P_TXZ][q] + ky * G[P_TYZ][q] + kz * G[P_TZZ][q])
                                  - I * kz * cs2 * S[F_RHO][q] - nu * k2 * G[P_UZ][q]);
                /* eq. (2): + f (steady body force; Fh is already masked) */
                if (c->Fh[0]) { R[F_MX][q] += c->Fh[0][q]; R[F_MY][q] += c->Fh[1][q]; R[F_MZ][q] += c->Fh[2][q]; }
                /* eq. (4): d B/dt = curl (u x B) + eta lap B */
                if (hydro) {
                    R[F_BX][q] = 0.0; R[F_BY][q] = 0.0; R[F_BZ][q] = 0.0;
                } else {
                    R[F_BX][q] = M * (I * (ky * G[P_EZ][q] - kz * G[P_EY][q])) - eta * k2 * S[F_BX][q];
                    R[F_BY][q] = M * (I * (kz * G[P_EX][q] - kx * G[P_EZ][q])) - eta * k2 * S[F_BY][q];
                    R[F_BZ][q] = M * (I * (kx * G[P_EY][q] - ky * G[P_EX][q])) - eta * k2 * S[F_BZ][q];
                }
            }
}

int mhd_ref_rhs(mhd_ref_ctx* c, double* out) {
    if (!c || !out) return MHD_REF_EINVAL;
    if (!c->have_fields) return MHD_REF_ESTATE;
    rhs(c, c->S, c->R);
    for (int i = 0; i < NFIELD; ++i) memcpy((cplx*)out + (size_t)i * c->nc, c->R[i], sizeof(cplx) * c->nc);
    return MHD_REF_OK;
}

/* a <- b + s*r over all fields and modes */
static void axpy_fields(const mhd_ref_ctx* c, cplx* const* a, cplx* const* b, double s, cplx* const* r) {
    for (int i = 0; i < NFIELD; ++i) {
        cplx* ai = a[i]; const cplx* bi = b[i]; const cplx* ri = r[i];
#pragma omp parallel for schedule(static)
        for (long long q = 0; q < (long long)c->nc; ++q) ai[q] = bi[q] + s * ri[q];
    }
}

/* step 3 of SURVEY.md §8(c.2) (AB2, Euler first step) and the classical RK4 of Table II */
int mhd_ref_step(mhd_ref_ctx* c, int nsteps) {
    if (!c || nsteps < 0) return MHD_REF_EINVAL;
    if (!c->have_fields) return MHD_REF_ESTATE;
    const double dt = c->dt;
    for (int n = 0; n < nsteps; ++n) {
        if (c->integrator == MHD_REF_AB2) {
            rhs(c, c->S, c->R);
            for (int i = 0; i < NFIELD; ++i) {
                cplx *S = c->S[i], *R = c->R[i], *Ro = c->Rold[i];
                const int hist = c->have_history;
#pragma omp parallel for schedule(static)
                for (long long q = 0; q < (long long)c->nc; ++q) {
                    if (hist) S[q] = S[q] + dt * (1.5 * R[q] - 0.5 * Ro[q]);
                    else      S[q] = S[q] + dt * R[q];
                    Ro[q] = R[q];
                }
            }
            c->have_history = 1;
        } else {
            /* k1..k4 with weights 1/6, 1/3, 1/3, 1/6 */
            for (int i = 0; i < NFIELD; ++i) memcpy(c->S0[i], c->S[i], sizeof(cplx) * c->nc);
            rhs(c, c->S, c->R);                                 /* k1 = R(S0) */
            axpy_fields(c, c->Acc, c->S0, dt / 6.0, c->R);
            axpy_fields(c, c->S, c->S0, 0.5 * dt, c->R);
            rhs(c, c->S, c->R);                                 /* k2 = R(S0 + dt/2 k1) */
            axpy_fields(c, c->Acc, c->Acc, dt / 3.0, c->R);
            axpy_fields(c, c->S, c->S0, 0.5 * dt, c->R);
            rhs(c, c->S, c->R);                                 /* k3 = R(S0 + dt/2 k2) */
            axpy_fields(c, c->Acc, c->Acc, dt / 3.0, c->R);
            axpy_fields(c, c->S, c->S0, dt, c->R);
            rhs(c, c->S, c->R);                                 /* k4 = R(S0 + dt k3) */
            axpy_fields(c, c->S, c->Acc, dt / 6.0, c->R);
        }
        c->step += 1;
        c->time += dt;
    }
    return MHD_REF_OK;
}

/* step 4 of SURVEY.md §8(c.2) */
int mhd_ref_get_fields(mhd_ref_ctx* c, double* rho, double* ux, double* uy, double* uz,
                       double* bx, double* by, double* bz) {
    if (!c || !rho || !ux || !uy || !uz) return MHD_REF_EINVAL;
    if (!c->have_fields) return MHD_REF_ESTATE;
    to_real(c, c->S);
    double* u[3] = {ux, uy, uz};
    double* b[3] = {bx, by, bz};
    memcpy(rho, c->f[F_RHO], sizeof(double) * c->nr);
    for (int i = 0; i < 3; ++i) {
        const double* m = c->f[F_MX + i];
        for (size_t p = 0; p < c->nr; ++p) u[i][p] = m[p] / rho[p];
        if (b[i]) memcpy(b[i], c->f[F_BX + i], sizeof(double) * c->nr);
    }
    return MHD_REF_OK;
}

int mhd_ref_get_spectral(mhd_ref_ctx* c, int field, double* out) {
    if (!c || !out || field < 0 || field >= NFIELD) return MHD_REF_EINVAL;
    memcpy(out, c->S[field], sizeof(cplx) * c->nc);
    return MHD_REF_OK;
}
int mhd_ref_set_spectral(mhd_ref_ctx* c, int field, const double* in) {
    if (!c || !in || field < 0 || field >= NFIELD) return MHD_REF_EINVAL;
    memcpy(c->S[field], in, sizeof(cplx) * c->nc);
    c->have_fields = 1;
    return MHD_REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * Diagnostics, SURVEY.md §8(c.2) step 5.  All averages are volume averages <.> = (1/N) sum_x.
 * Sums are serial Neumaier-compensated, so they are order-fixed and accurate to ~1 ulp.
 * ------------------------------------------------------------------------------------------ */
typedef struct { double s, c; } ksum;
static void ksum_add(ksum* k, double v) {
    double t = k->s + v;
    if (fabs(k->s) >= fabs(v)) k->c += (k->s - t) + v; else k->c += (v - t) + k->s;
    k->s = t;
}
static double ksum_get(const ksum* k) { return k->s + k->c; }

static int shell_of(double k2) { return (int)floor(sqrt(k2) + 0.5); }

int mhd_ref_diagnostics(mhd_ref_ctx* c, mhd_ref_diag* d, double* ekin_spec, double* emag_spec, int nshell) {
    if (!c || !d || nshell < 0 || (nshell > 0 && (!ekin_spec || !emag_spec))) return MHD_REF_EINVAL;
    if (!c->have_fields) return MHD_REF_ESTATE;
    const double Ninv = 1.0 / (double)c->nr;
    int bad = 0;
    to_real(c, c->S);
    ksum ek = {0, 0}, em = {0, 0}, ei = {0, 0}, ma = {0, 0}, mo[3] = {{0, 0}, {0, 0}, {0, 0}}, bm[3] = {{0, 0}, {0, 0}, {0, 0}};
    for (size_t p = 0; p < c->nr; ++p) {
        double rho = c->f[F_RHO][p];
        double mx = c->f[F_MX][p], my = c->f[F_MY][p], mz = c->f[F_MZ][p];
        double bx = c->f[F_BX][p], by = c->f[F_BY][p], bz = c->f[F_BZ][p];
        if (!(rho > 0.0) || !isfinite(rho) || !isfinite(mx) || !isfinite(my) || !isfinite(mz) ||
            !isfinite(bx) || !isfinite(by) || !isfinite(bz)) bad = 1;
        ksum_add(&ek, 0.5 * (mx * mx + my * my + mz * mz) / rho);   /* 1/2 rho |u|^2 = 1/2 m.u */
        ksum_add(&em, 0.5 * (bx * bx + by * by + bz * bz));          /* 1/2 |B|^2  */
        ksum_add(&ei, rho * log(rho));
        ksum_add(&ma, rho);
        ksum_add(&mo[0], mx); ksum_add(&mo[1], my); ksum_add(&mo[2], mz);
        ksum_add(&bm[0], bx); ksum_add(&bm[1], by); ksum_add(&bm[2], bz);
    }
    d->step = c->step; d->time = c->time;
    d->ekin = ksum_get(&ek) * Ninv; d->emag = ksum_get(&em) * Ninv;
    d->eiso = c->cs * c->cs * ksum_get(&ei) * Ninv; d->mass = ksum_get(&ma) * Ninv;
    for (int i = 0; i < 3; ++i) { d->mom[i] = ksum_get(&mo[i]) * Ninv; d->bmean[i] = ksum_get(&bm[i]) * Ninv; }

    /* max_x |IFFT(i k.B^)| */
    for (int jz = 0; jz < c->nz; ++jz)
        for (int jy = 0; jy < c->ny; ++jy)
            for (int jx = 0; jx < c->nxh; ++jx) {
                size_t q = ((size_t)jz * c->ny + jy) * c->nxh + jx;
                double kx = c->kfac[0] * jx, ky = c->kfac[1] * wavenumber(jy, c->ny), kz = c->kfac[2] * wavenumber(jz, c->nz);
                c->tmp[q] = I * (kx * c->S[F_BX][q] + ky * c->S[F_BY][q] + kz * c->S[F_BZ][q]);
            }
    c2r3(&c->plan, c->tmp, c->g[0]);
    double mx = 0.0;
    for (size_t p = 0; p < c->nr; ++p) { double a = fabs(c->g[0][p]); if (a > mx) mx = a; if (!isfinite(a)) bad = 1; }
    d->max_divb = mx;

    /* u^ = FFT(m/rho) over EVERY mode (u is not band-limited): needed by the paper diagnostics and the spectra */
    to_real(c, c->S);
    for (int i = 0; i < 3; ++i) {
        for (size_t p = 0; p < c->nr; ++p) c->g[i][p] = c->f[F_MX + i][p] / c->f[F_RHO][p];
        r2c3(&c->plan, c->g[i], c->G[i]);
    }
    /* Omega(t) = <|curl u|^2>, <|curl B|^2>, <|u|^2>, Rayleigh quotient eq. (14), as
     * sums over the full spectrum (Parseval): half-spectrum entries with 0 < kx < nx/2 stand for two modes. */
    {
        ksum en = {0, 0}, cu = {0, 0}, u2 = {0, 0};
        for (int jz = 0; jz < c->nz; ++jz)
            for (int jy = 0; jy < c->ny; ++jy)
                for (int jx = 0; jx < c->nxh; ++jx) {
                    size_t q = ((size_t)jz * c->ny + jy) * c->nxh + jx;
                    double kx = c->kfac[0] * jx, ky = c->kfac[1] * wavenumber(jy, c->ny), kz = c->kfac[2] * wavenumber(jz, c->nz);
                    double w = (jx == 0 || 2 * jx == c->nx) ? 1.0 : 2.0;
                    cplx ux = c->G[0][q], uy = c->G[1][q], uz = c->G[2][q];
                    cplx wx = ky * uz - kz * uy, wy = kz * ux - kx * uz, wz = kx * uy - ky * ux;      /* (k x u^) */
                    ksum_add(&en, w * (creal(wx) * creal(wx) + cimag(wx) * cimag(wx) + creal(wy) * creal(wy) + cimag(wy) * cimag(wy) +
                                       creal(wz) * creal(wz) + cimag(wz) * cimag(wz)));
                    ksum_add(&u2, w * (creal(ux) * creal(ux) + cimag(ux) * cimag(ux) + creal(uy) * creal(uy) + cimag(uy) * cimag(uy) +
                                       creal(uz) * creal(uz) + cimag(uz) * cimag(uz)));
                    cplx bx = c->S[F_BX][q], by = c->S[F_BY][q], bz = c->S[F_BZ][q];
                    cplx jx_ = ky * bz - kz * by, jy_ = kz * bx - kx * bz, jz_ = kx * by - ky * bx;   /* (k x B^) */
                    ksum_add(&cu, w * (creal(jx_) * creal(jx_) + cimag(jx_) * cimag(jx_) + creal(jy_) * creal(jy_) + cimag(jy_) * cimag(jy_) +
                                       creal(jz_) * creal(jz_) + cimag(jz_) * cimag(jz_)));
                }
        d->enstrophy = ksum_get(&en) * Ninv * Ninv;
        d->current2 = ksum_get(&cu) * Ninv * Ninv;
        d->u2 = ksum_get(&u2) * Ninv * Ninv;
        double den = d->u2 + d->emag;                 /* <|u|^2> + 1/2 <|B|^2>,  emag = 1/2 <|B|^2> */
        d->rayleigh_q = den > 0.0 ? (d->enstrophy + 0.5 * d->current2) / den : 0.0;
    }

    /* shell spectra: s = round(|k|); velocity power 1/2|u^|^2/N^2 (u = m/rho, not density weighted),
     * magnetic power 1/2|B^|^2/N^2; half-spectrum entries with 0 < kx < nx/2 stand for two modes. */
    if (nshell > 0) {
        if (c->kfac[0] != 1.0 || c->kfac[1] != 1.0 || (c->nz > 1 && c->kfac[2] != 1.0)) return MHD_REF_EINVAL;   /* 2*pi box only */
        ksum* ks = (ksum*)calloc((size_t)nshell * 2, sizeof(ksum));
        if (!ks) return MHD_REF_ENOMEM;
        for (int jz = 0; jz < c->nz; ++jz)
            for (int jy = 0; jy < c->ny; ++jy)
                for (int jx = 0; jx < c->nxh; ++jx) {
                    size_t q = ((size_t)jz * c->ny + jy) * c->nxh + jx;
                    double kx = jx, ky = wavenumber(jy, c->ny), kz = wavenumber(jz, c->nz);
                    int s = shell_of(kx * kx + ky * ky + kz * kz);
                    if (s >= nshell) continue;
                    double w = (jx == 0 || 2 * jx == c->nx) ? 1.0 : 2.0;
                    double pu = 0.0, pb = 0.0;
                    for (int i = 0; i < 3; ++i) {
                        cplx u = c->G[i][q], b = c->S[F_BX + i][q];
                        pu += creal(u) * creal(u) + cimag(u) * cimag(u);
                        pb += creal(b) * creal(b) + cimag(b) * cimag(b);
                    }
                    ksum_add(&ks[s], 0.5 * w * pu);
                    ksum_add(&ks[nshell + s], 0.5 * w * pb);
                }
        for (int s = 0; s < nshell; ++s) {
            ekin_spec[s] = ksum_get(&ks[s]) * Ninv * Ninv;
            emag_spec[s] = ksum_get(&ks[nshell + s]) * Ninv * Ninv;
        }
        free(ks);
    }
    return bad ? MHD_REF_ENONFINITE : MHD_REF_OK;
}
