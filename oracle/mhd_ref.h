/* mhd_ref.h — CPU ORACLE for the pseudo-spectral isothermal MHD step.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct restatement of the method of arxiv 2402.05478:
 *   eqs (1)-(4), PAPER.md:39-47        continuity, momentum, isothermal EOS, induction
 *   "pseudo-spectral ... 2/3 de-aliasing rule ... Adams-bashforth"
 *   "Time integration: Adams-Bashforth, Runge-Kutta 4", PAPER.md:105 (Table II)
 *   "Precision: Double"
 * following SURVEY.md §8(c.2) step by step, with its own recursive FFT.  All pointers are HOST
 * pointers.  It shares no code with the CUDA library (include/mhd.h, paper_2402_05478_b200/csrc).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it; the product path never does.
 *
 * Parity pins (tests/test_oracle_*.py): brute-force DFT, numpy.fft, exact single-mode viscous /
 * resistive decay, circularly polarised Alfven wave (sign of eq. 4), sound / fast-wave frequency,
 * exact invariants, div B at roundoff, ideal-limit energy drift order, energy balance, cyclic
 * axis permutation, KH linear growth; box lengths by the exact rescaling x -> 2*pi*x/L of the
 * equations; forcing by the exact forced shear-wave recurrence and the momentum budget; enstrophy /
 * Rayleigh quotient by Beltrami (curl u = k0 u) closed forms and a numpy restatement.  PARITY UNPINNED by the paper (API definitions fixed by
 * SURVEY.md §8(c.3), not by PAPER.md): the order of the Adams-Bashforth scheme (AB2 with an Euler
 * first step), the sound speed of each config, and the definition of the shell spectra.
 *
 * Layouts.  Real fields: [nz][ny][nx] doubles, x fastest.  Half-spectra: [nz][ny][nx/2+1]
 * complex (re,im interleaved), kx = 0..nx/2 fastest, ky and kz in FFT order (0..n/2-1, -n/2..-1).
 * Forward DFT  f^(k) = sum_x f(x) exp(-i k.x)  (unnormalised); inverse divides by nx*ny*nz.
 */
#ifndef MHD_REF_H
#define MHD_REF_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mhd_ref_ctx mhd_ref_ctx;

enum { MHD_REF_OK = 0, MHD_REF_EINVAL = -1, MHD_REF_ENOMEM = -2, MHD_REF_ESTATE = -4, MHD_REF_ENONFINITE = -5 };
enum { MHD_REF_AB2 = 0, MHD_REF_RK4 = 1 };
enum { MHD_REF_FLAG_HYDRO = 1u, MHD_REF_FLAG_NO_DEALIAS = 2u };

typedef struct {
    long long step;
    double time, ekin, emag, eiso, mass, mom[3], bmean[3], max_divb;
    /* paper diagnostics, all from the spectra of u = m/rho (every mode) and B:
     *   enstrophy  = <|curl u|^2> = sum_k |k x u^(k)|^2 / N^2      Omega(t)
     *   current2   = <|curl B|^2> = sum_k |k x B^(k)|^2 / N^2
     *   u2         = <|u|^2>      = sum_k |u^(k)|^2 / N^2
     *   rayleigh_q = (enstrophy + current2/2) / (u2 + <|B|^2>/2)     eq. (14) */
    double enstrophy, current2, u2, rayleigh_q;
} mhd_ref_diag;

/* threads used by the row loops (OpenMP); results do not depend on it */
void mhd_ref_set_threads(int n);
int  mhd_ref_get_threads(void);

/* 1-D complex DFT of length n (any n >= 1), sign = -1 forward, +1 inverse (unnormalised). */
int mhd_ref_fft1d(int n, int sign, const double* in_complex, double* out_complex);
/* batched 3-D real-to-complex (unnormalised) and complex-to-real (includes 1/(nx ny nz)). */
int mhd_ref_fft_r2c(int nx, int ny, int nz, int batch, const double* in_real, double* out_complex);
int mhd_ref_fft_c2r(int nx, int ny, int nz, int batch, const double* in_complex, double* out_real);

int  mhd_ref_create(mhd_ref_ctx** out, int nx, int ny, int nz, double nu, double eta, double cs, double dt,
                    int integrator, unsigned flags);
void mhd_ref_destroy(mhd_ref_ctx*);
/* Box lengths (the KH test uses Lx = 1, Ly = 2): wavenumbers become k_i = 2*pi*n_i/L_i.
 * Default 2*pi per axis (k = n exactly).  The 2/3 mask stays a test on the integer n_i.  lz is ignored
 * when nz == 1.  Shell spectra are defined for the 2*pi box only. */
int  mhd_ref_set_box(mhd_ref_ctx*, double lx, double ly, double lz);
/* Steady body force f(x) of eq. (2) ("+ f"; App. B eqs B2-B3): its masked
 * transform is added to the momentum right-hand side.  NULL, NULL, NULL switches it off. */
int  mhd_ref_set_forcing(mhd_ref_ctx*, const double* fx, const double* fy, const double* fz);
int  mhd_ref_set_fields(mhd_ref_ctx*, const double* rho, const double* ux, const double* uy, const double* uz,
                        const double* bx, const double* by, const double* bz);
int  mhd_ref_step(mhd_ref_ctx*, int nsteps);
int  mhd_ref_get_fields(mhd_ref_ctx*, double* rho, double* ux, double* uy, double* uz,
                        double* bx, double* by, double* bz);
int  mhd_ref_diagnostics(mhd_ref_ctx*, mhd_ref_diag* out, double* ekin_spec, double* emag_spec, int nshell);

/* test hooks: the spectral state (field 0..6 = rho^, mx^, my^, mz^, Bx^, By^, Bz^) and the
 * right-hand side R(S) of the current state, both as full half-spectra. */
int mhd_ref_get_spectral(mhd_ref_ctx*, int field, double* out_complex);
int mhd_ref_set_spectral(mhd_ref_ctx*, int field, const double* in_complex);
int mhd_ref_rhs(mhd_ref_ctx*, double* out_complex_7_fields);
/* the de-aliasing mask M(k) as 0/1 bytes over the half-spectrum */
int mhd_ref_mask(mhd_ref_ctx*, unsigned char* out);

#ifdef __cplusplus
}
#endif
#endif
