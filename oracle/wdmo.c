/*
 * wdmo.c -- CPU ORACLE for the split-step Schroedinger-Poisson + CIC particle step.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call this file.  It is
 * plain, slow, float64 C written from the paper, shares no code with the CUDA path
 * (paper_2606_25026_b200/csrc/) and is never tuned.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md at authoring time):
 *   - kick-drift-kick split step, Eq. 16-18 and Algorithm 1 lines 5-16
 *     (PAPER.md:247-267): (a) psi *= exp(-i Phi dt/(2 mu)), (b) psi = F^-1{exp(-i mu k^2 dt/2) F{psi}},
 *     (c) Phi = F^-1{-4 pi G rho_k / k^2}, k = 0 mode zeroed (Eq. 23), (d) second half kick
 *     with the NEW Phi.  mu = hbar/m; |psi|^2 is mass density (reading G6).
 *   - grid x_i = -L/2 + i dx (Eq. 20) with dx = L/N (reading G1, periodic box).
 *   - particles: "N-body particles contribute their gravitational potential to the grid ... the wave
 *     dark matter gravitational acceleration is interpolated from the grid to particle positions"
 *     (PAPER.md:314); realised, as BASELINE.json's north_star prescribes, by a cloud-in-cell deposit into
 *     the Poisson source, a 2nd-order central-difference gradient (Eq. 21) gathered with
 *     the same CIC weights, and a kick-drift-kick leapfrog sharing dt (readings G11-G16).
 *   - the absorbing mask of Alg. 1 l.17-18 is NOT applied (reading G10; Eq. 22 is garbled).
 *   - the 3-D DFT is separable; each 1-D transform is the textbook recursive radix-2
 *     decimation-in-time FFT below; forward kernel e^{-ikx}, inverse carries 1/N per axis (reading G7).
 *     A direct O(n^2) DFT is exported for the brute-force pin (tests/test_oracle_pins.py P5).
 *
 * Pins (tests/test_oracle_pins.py): P1 norm, P2 free Gaussian closed form, P3 plane wave,
 * P4 single-mode Poisson, P5 direct DFT, P6 O(dt^2) energy error, P7 time reversal, P8 CIC
 * momentum / mass / zero self force, P9 gather in a known field, P10 numpy.fft cross-check.
 * P11 self-interaction plane wave, P12 external potential (harmonic ground state, particles feel it), P13 absorbing-layer
 * values at face / edge / corner, P14 diagnostics closed forms (plane wave, real Gaussian, cosine density, Eq. 26),
 * P15 sub-stepped leapfrog in a harmonic potential / static particles.
 * P16 triangular-shaped cloud: hand-computed weights, mass / centre / second moment, exact gradient of a
 * quadratic-free (single-mode) field, momentum conservation.
 * P17 spectral kinetic energy (plane-wave closed forms incl. a Nyquist component, T -> K + Q at second order in dx, the
 * moving-Gaussian closed form), E = T + W against numpy.fft and its O(dt^2) drift, the per-step record against a
 * hand-undone closing kick; the density getter with an absorbing layer (reading G22).
 * The coupled psi+particle trajectory over many steps has no closed form: "parity unpinned"
 * beyond P1, P7, P8 and second-order self-convergence.
 *
 * Threads: OpenMP over pencils / particles where the loop iterations are independent; the CIC
 * deposit is serial (it is a scatter-add).  No blocking, fusion or reordering.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

enum { WDMO_OK = 0, WDMO_EINVAL = 1, WDMO_EUNSUPPORTED = 2, WDMO_ENOMEM = 3, WDMO_ESTATE = 5 };

typedef struct wdmo_ctx {
    int N;
    double L, mu, G, dx;
    size_t n;            /* N^3 */
    cplx *psi;           /* N^3, C order (ix, iy, iz), iz contiguous */
    cplx *work;          /* N^3 scratch */
    double *rho, *phi;   /* N^3 */
    long long np;
    double *pos, *vel, *acc, *mass; /* np x 3, np */
    int have_psi, stale;
    /* extra kick terms (Eq. 13-14, Eq. 22, Alg. 1 l.15-18; readings G26-G28) */
    double kappa;        /* local self-interaction: V += kappa |psi|^2                         */
    double *phi_ext;     /* static external potential added to the Poisson potential, or NULL  */
    double alpha;        /* absorbing-layer coefficient (0 = no layer)                          */
    int nb;              /* absorbing-layer transition width L / nb                             */
    /* particle variants (reading G29) */
    int nsub;            /* leapfrog sub-steps per SPE step (>= 1)                              */
    int pstatic;         /* :particles_static -- particles never move, they only source Phi    */
    int order;           /* mass assignment / force interpolation: 2 = cloud-in-cell, 3 = TSC   */
    /* per-step diagnostics, recorded between (c) and (d) of the last step when switched on */
    int step_diag_on, step_diag_valid;
    double step_diag[8];
    double *phi_grav;    /* Poisson potential before Phi_ext is added (only kept while step_diag_on)          */
} wdmo_ctx;

static int is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

/* ---------------------------------------------------------------- 1-D transforms */

/* Direct DFT: out[k] = sum_j in[j] exp(sign * 2 pi i j k / n).  O(n^2), any n. */
static void dft_direct(const cplx *in, cplx *out, int n, int sign)
{
    for (int k = 0; k < n; ++k) {
        cplx s = 0.0;
        for (int j = 0; j < n; ++j) {
            double a = sign * 2.0 * M_PI * (double)(((long long)j * k) % n) / (double)n;
            s += in[j] * (cos(a) + I * sin(a));
        }
        out[k] = s;
    }
}

/* Textbook recursive radix-2 decimation-in-time FFT.  tw[j] = exp(sign 2 pi i j / n_full);
 * for a sub-transform of length n the twiddle w_n^k is tw[k * twstep], twstep = n_full / n. */
static void fft_rec(const cplx *in, int stride, cplx *out, int n, const cplx *tw, int twstep)
{
    if (n == 1) { out[0] = in[0]; return; }
    int h = n / 2;
    fft_rec(in, 2 * stride, out, h, tw, 2 * twstep);              /* even samples */
    fft_rec(in + stride, 2 * stride, out + h, h, tw, 2 * twstep); /* odd samples  */
    for (int k = 0; k < h; ++k) {
        cplx e = out[k], t = tw[k * twstep] * out[k + h];
        out[k] = e + t;
        out[k + h] = e - t;
    }
}

static cplx *make_twiddles(int n, int sign)
{
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)(n > 1 ? n : 1));
    if (!tw) return NULL;
    for (int j = 0; j < n; ++j) {
        double a = sign * 2.0 * M_PI * (double)j / (double)n;
        tw[j] = cos(a) + I * sin(a);
    }
    return tw;
}

/* sign = -1 forward (unnormalised), +1 inverse (times 1/n). */
int wdmo_fft1d(int n, const double *in, double *out, int sign)
{
    if (!is_pow2(n) || !in || !out || (sign != 1 && sign != -1)) return WDMO_EINVAL;
    cplx *tw = make_twiddles(n, sign);
    if (!tw) return WDMO_ENOMEM;
    fft_rec((const cplx *)in, 1, (cplx *)out, n, tw, 1);
    if (sign == 1) for (int j = 0; j < n; ++j) ((cplx *)out)[j] /= (double)n;
    free(tw);
    return WDMO_OK;
}

int wdmo_dft1d_direct(int n, const double *in, double *out, int sign)
{
    if (n < 1 || !in || !out || (sign != 1 && sign != -1)) return WDMO_EINVAL;
    dft_direct((const cplx *)in, (cplx *)out, n, sign);
    if (sign == 1) for (int j = 0; j < n; ++j) ((cplx *)out)[j] /= (double)n;
    return WDMO_OK;
}

/* ---------------------------------------------------------------- 3-D transforms */

/* In-place separable 3-D DFT of a[N][N][N]: one 1-D transform along every pencil of each axis. */
static int fft3_inplace(cplx *a, int N, int sign)
{
    cplx *tw = make_twiddles(N, sign);
    if (!tw) return WDMO_ENOMEM;
    size_t N2 = (size_t)N * N;
    int fail = 0;
    for (int axis = 2; axis >= 0; --axis) {
        size_t st = axis == 2 ? 1 : (axis == 1 ? (size_t)N : N2);        /* stride along the axis */
#pragma omp parallel
        {
            cplx *line = (cplx *)malloc(sizeof(cplx) * 2 * (size_t)N);
            if (!line) {
#pragma omp atomic write
                fail = 1;
            }
#pragma omp for schedule(static)
            for (long long p = 0; p < (long long)N2; ++p) {
                if (!line) continue;
                size_t u = (size_t)p / N, v = (size_t)p % N, base;     /* the two other indices */
                if (axis == 2) base = u * N2 + v * N;                    /* (ix=u, iy=v, :)  */
                else if (axis == 1) base = u * N2 + v;                   /* (ix=u, :, iz=v)  */
                else base = u * N + v;                                   /* (:, iy=u, iz=v)  */
                cplx *in = line, *out = line + N;
                for (int j = 0; j < N; ++j) in[j] = a[base + j * st];
                fft_rec(in, 1, out, N, tw, 1);
                if (sign == 1) for (int j = 0; j < N; ++j) a[base + j * st] = out[j] / (double)N;
                else for (int j = 0; j < N; ++j) a[base + j * st] = out[j];
            }
            free(line);
        }
    }
    free(tw);
    return fail ? WDMO_ENOMEM : WDMO_OK;
}

int wdmo_fft3(int N, const double *in, double *out, int sign)
{
    if (!is_pow2(N) || !in || !out || (sign != 1 && sign != -1)) return WDMO_EINVAL;
    size_t n = (size_t)N * N * N;
    if (in != out) memcpy(out, in, sizeof(cplx) * n);
    return fft3_inplace((cplx *)out, N, sign);
}

/* Brute force: out[k] = sum_j in[j] exp(sign 2 pi i (j.k)/N), the plain triple sum.  O(N^6). */
int wdmo_dft3_direct(int N, const double *in_, double *out_, int sign)
{
    if (N < 1 || N > 16 || !in_ || !out_ || (sign != 1 && sign != -1)) return WDMO_EINVAL;
    const cplx *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
    for (int kx = 0; kx < N; ++kx) for (int ky = 0; ky < N; ++ky) for (int kz = 0; kz < N; ++kz) {
        cplx s = 0.0;
        for (int jx = 0; jx < N; ++jx) for (int jy = 0; jy < N; ++jy) for (int jz = 0; jz < N; ++jz) {
            long long m = ((long long)jx * kx + (long long)jy * ky + (long long)jz * kz) % N;
            double a = sign * 2.0 * M_PI * (double)m / (double)N;
            s += in[((size_t)jx * N + jy) * N + jz] * (cos(a) + I * sin(a));
        }
        if (sign == 1) s /= (double)N * N * N;
        out[((size_t)kx * N + ky) * N + kz] = s;
    }
    return WDMO_OK;
}

/* signed wavenumber k = 2 pi s(j) / L, s(j) = j for j < N/2 else j - N (reading G4) */
static double wavenumber(int j, int N, double L)
{
    int s = j < N / 2 ? j : j - N;
    if (N == 1) s = 0;
    return 2.0 * M_PI * (double)s / L;
}

/* ---------------------------------------------------------------- Poisson (Eq. 18c, Eq. 23) */

/* phi = Re F^-1{ -4 pi G rho_k / k^2 }, rho_k(k=0) dropped  ( == subtracting <rho>, reading G3 ). */
static int poisson(const double *rho, double *phi, cplx *work, int N, double L, double G)
{
    size_t n = (size_t)N * N * N;
    for (size_t i = 0; i < n; ++i) work[i] = rho[i];
    int rc = fft3_inplace(work, N, -1);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int ix = 0; ix < N; ++ix) {
        double kx = wavenumber(ix, N, L);
        for (int iy = 0; iy < N; ++iy) {
            double ky = wavenumber(iy, N, L);
            for (int iz = 0; iz < N; ++iz) {
                double kz = wavenumber(iz, N, L);
                double k2 = kx * kx + ky * ky + kz * kz;
                size_t i = ((size_t)ix * N + iy) * N + iz;
                if (ix == 0 && iy == 0 && iz == 0) work[i] = 0.0;
                else work[i] *= -4.0 * M_PI * G / k2;
            }
        }
    }
    rc = fft3_inplace(work, N, +1);
    if (rc) return rc;
    for (size_t i = 0; i < n; ++i) phi[i] = creal(work[i]);
    return WDMO_OK;
}

int wdmo_poisson(int N, double L, double G, const double *rho, double *phi)
{
    if (!is_pow2(N) || L <= 0 || !rho || !phi) return WDMO_EINVAL;
    cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)N * N * N);
    if (!work) return WDMO_ENOMEM;
    int rc = poisson(rho, phi, work, N, L, G);
    free(work);
    return rc;
}

/* ---------------------------------------------------------------- cloud-in-cell (readings G12, G13) */

static int wrap_index(long long i, int N) { long long r = i % N; return (int)(r < 0 ? r + N : r); }

/* rho[(i0 + corner) mod N] += m w / dx^3 for the 8 nodes around each particle; u = (x + L/2)/dx,
 * i0 = floor(u), f = u - i0, w = prod_axis (f if corner bit else 1 - f).  Adds into rho. */
static void cic_deposit(double *rho, int N, double L, long long np, const double *pos,
                        const double *mass)
{
    double dx = L / N, inv_vol = 1.0 / (dx * dx * dx);
    for (long long p = 0; p < np; ++p) {
        long long i0[3]; double f[3];
        for (int a = 0; a < 3; ++a) {
            double u = (pos[3 * p + a] + 0.5 * L) / dx;
            double fl = floor(u);
            i0[a] = (long long)fl;
            f[a] = u - fl;
        }
        for (int c = 0; c < 8; ++c) {
            int bx = (c >> 2) & 1, by = (c >> 1) & 1, bz = c & 1;
            double w = (bx ? f[0] : 1.0 - f[0]) * (by ? f[1] : 1.0 - f[1]) * (bz ? f[2] : 1.0 - f[2]);
            size_t idx = ((size_t)wrap_index(i0[0] + bx, N) * N + wrap_index(i0[1] + by, N)) * N
                         + wrap_index(i0[2] + bz, N);
            rho[idx] += mass[p] * w * inv_vol;
        }
    }
}

/* g_axis[node] = -(phi[node + e_axis] - phi[node - e_axis]) / (2 dx)  (Eq. 21), then
 * a_axis(x_p) = sum_corners w g_axis[(i0 + corner) mod N] with the deposit's weights. */
static void cic_gather(const double *phi, int N, double L, long long np, const double *pos, double *acc)
{
    double dx = L / N;
#pragma omp parallel for schedule(static)
    for (long long p = 0; p < np; ++p) {
        long long i0[3]; double f[3];
        for (int a = 0; a < 3; ++a) {
            double u = (pos[3 * p + a] + 0.5 * L) / dx;
            double fl = floor(u);
            i0[a] = (long long)fl;
            f[a] = u - fl;
        }
        double ax = 0.0, ay = 0.0, az = 0.0;
        for (int c = 0; c < 8; ++c) {
            int bx = (c >> 2) & 1, by = (c >> 1) & 1, bz = c & 1;
            double w = (bx ? f[0] : 1.0 - f[0]) * (by ? f[1] : 1.0 - f[1]) * (bz ? f[2] : 1.0 - f[2]);
            int ix = wrap_index(i0[0] + bx, N), iy = wrap_index(i0[1] + by, N), iz = wrap_index(i0[2] + bz, N);
#define PHI(a, b, c_) phi[((size_t)wrap_index((a), N) * N + wrap_index((b), N)) * N + wrap_index((c_), N)]
            ax += w * -(PHI(ix + 1, iy, iz) - PHI(ix - 1, iy, iz)) / (2.0 * dx);
            ay += w * -(PHI(ix, iy + 1, iz) - PHI(ix, iy - 1, iz)) / (2.0 * dx);
            az += w * -(PHI(ix, iy, iz + 1) - PHI(ix, iy, iz - 1)) / (2.0 * dx);
#undef PHI
        }
        acc[3 * p] = ax; acc[3 * p + 1] = ay; acc[3 * p + 2] = az;
    }
}

int wdmo_cic_deposit(int N, double L, long long np, const double *pos, const double *mass, double *rho)
{
    if (N < 1 || L <= 0 || np < 0 || !rho || (np > 0 && (!pos || !mass))) return WDMO_EINVAL;
    cic_deposit(rho, N, L, np, pos, mass);
    return WDMO_OK;
}

int wdmo_cic_gather(int N, double L, const double *phi, long long np, const double *pos, double *acc)
{
    if (N < 1 || L <= 0 || np < 0 || !phi || (np > 0 && (!pos || !acc))) return WDMO_EINVAL;
    cic_gather(phi, N, L, np, pos, acc);
    return WDMO_OK;
}

/* ---------------------------------------------------------------- triangular-shaped cloud (reading G30)
 *
 * Second-order assignment (Hockney & Eastwood, "Computer Simulation Using Particles", sec. 5-2-4): with
 * u = (x + L/2)/dx, j = floor(u + 1/2) the NEAREST node and d = u - j in [-1/2, 1/2), the particle's mass goes
 * to the three nodes j-1, j, j+1 per axis with weights
 *      w(-1) = (1/2 - d)^2 / 2,    w(0) = 3/4 - d^2,    w(+1) = (1/2 + d)^2 / 2
 * (the overlap of a triangle of base 2 dx centred on the particle with each node's cell); 27 nodes in 3-D, the
 * weight the product over axes.  The gather uses the same weights on the same central-difference gradient as G13. */

static void tsc_weights(double x, double L, double dx, long long *j, double w[3])
{
    double u = (x + 0.5 * L) / dx;
    double fl = floor(u + 0.5);
    double d = u - fl;
    *j = (long long)fl;
    w[0] = 0.5 * (0.5 - d) * (0.5 - d);
    w[1] = 0.75 - d * d;
    w[2] = 0.5 * (0.5 + d) * (0.5 + d);
}

static void tsc_deposit(double *rho, int N, double L, long long np, const double *pos, const double *mass)
{
    double dx = L / N, inv_vol = 1.0 / (dx * dx * dx);
    for (long long p = 0; p < np; ++p) {
        long long j[3]; double w[3][3];
        for (int a = 0; a < 3; ++a) tsc_weights(pos[3 * p + a], L, dx, &j[a], w[a]);
        for (int ox = -1; ox <= 1; ++ox)
            for (int oy = -1; oy <= 1; ++oy)
                for (int oz = -1; oz <= 1; ++oz) {
                    size_t idx = ((size_t)wrap_index(j[0] + ox, N) * N + wrap_index(j[1] + oy, N)) * N
                                 + wrap_index(j[2] + oz, N);
                    rho[idx] += mass[p] * w[0][ox + 1] * w[1][oy + 1] * w[2][oz + 1] * inv_vol;
                }
    }
}

static void tsc_gather(const double *phi, int N, double L, long long np, const double *pos, double *acc)
{
    double dx = L / N;
#pragma omp parallel for schedule(static)
    for (long long p = 0; p < np; ++p) {
        long long j[3]; double w[3][3];
        for (int a = 0; a < 3; ++a) tsc_weights(pos[3 * p + a], L, dx, &j[a], w[a]);
        double ax = 0.0, ay = 0.0, az = 0.0;
        for (int ox = -1; ox <= 1; ++ox)
            for (int oy = -1; oy <= 1; ++oy)
                for (int oz = -1; oz <= 1; ++oz) {
                    double wt = w[0][ox + 1] * w[1][oy + 1] * w[2][oz + 1];
                    long long ix = j[0] + ox, iy = j[1] + oy, iz = j[2] + oz;
#define PHI(a, b, c_) phi[((size_t)wrap_index((a), N) * N + wrap_index((b), N)) * N + wrap_index((c_), N)]
                    ax += wt * -(PHI(ix + 1, iy, iz) - PHI(ix - 1, iy, iz)) / (2.0 * dx);
                    ay += wt * -(PHI(ix, iy + 1, iz) - PHI(ix, iy - 1, iz)) / (2.0 * dx);
                    az += wt * -(PHI(ix, iy, iz + 1) - PHI(ix, iy, iz - 1)) / (2.0 * dx);
#undef PHI
                }
        acc[3 * p] = ax; acc[3 * p + 1] = ay; acc[3 * p + 2] = az;
    }
}

int wdmo_tsc_deposit(int N, double L, long long np, const double *pos, const double *mass, double *rho)
{
    if (N < 1 || L <= 0 || np < 0 || !rho || (np > 0 && (!pos || !mass))) return WDMO_EINVAL;
    tsc_deposit(rho, N, L, np, pos, mass);
    return WDMO_OK;
}

int wdmo_tsc_gather(int N, double L, const double *phi, long long np, const double *pos, double *acc)
{
    if (N < 1 || L <= 0 || np < 0 || !phi || (np > 0 && (!pos || !acc))) return WDMO_EINVAL;
    tsc_gather(phi, N, L, np, pos, acc);
    return WDMO_OK;
}

/* the context's scheme */
static void assign_deposit(const wdmo_ctx *c, double *rho)
{
    if (c->order == 3) tsc_deposit(rho, c->N, c->L, c->np, c->pos, c->mass);
    else cic_deposit(rho, c->N, c->L, c->np, c->pos, c->mass);
}

static void assign_gather(wdmo_ctx *c)
{
    if (c->order == 3) tsc_gather(c->phi, c->N, c->L, c->np, c->pos, c->acc);
    else cic_gather(c->phi, c->N, c->L, c->np, c->pos, c->acc);
}

/* ---------------------------------------------------------------- context */

int wdmo_create(wdmo_ctx **out, int N, double L, double hbar_over_m, double G)
{
    if (!out) return WDMO_EINVAL;
    *out = NULL;
    if (!(L > 0) || !(hbar_over_m > 0) || !(G >= 0)) return WDMO_EINVAL;
    if (!is_pow2(N) || N < 2 || N > 1024) return WDMO_EUNSUPPORTED;
    wdmo_ctx *c = (wdmo_ctx *)calloc(1, sizeof(*c));
    if (!c) return WDMO_ENOMEM;
    c->N = N; c->L = L; c->mu = hbar_over_m; c->G = G; c->dx = L / N;
    c->nsub = 1;
    c->order = 2;
    c->n = (size_t)N * N * N;
    c->psi = (cplx *)malloc(sizeof(cplx) * c->n);
    c->work = (cplx *)malloc(sizeof(cplx) * c->n);
    c->rho = (double *)malloc(sizeof(double) * c->n);
    c->phi = (double *)malloc(sizeof(double) * c->n);
    if (!c->psi || !c->work || !c->rho || !c->phi) {
        free(c->psi); free(c->work); free(c->rho); free(c->phi); free(c);
        return WDMO_ENOMEM;
    }
    c->stale = 1;
    *out = c;
    return WDMO_OK;
}

int wdmo_destroy(wdmo_ctx *c)
{
    if (!c) return WDMO_OK;
    free(c->psi); free(c->work); free(c->rho); free(c->phi);
    free(c->pos); free(c->vel); free(c->acc); free(c->mass);
    free(c->phi_ext); free(c->phi_grav);
    free(c);
    return WDMO_OK;
}

int wdmo_set_psi(wdmo_ctx *c, const double *psi)
{
    if (!c || !psi) return WDMO_EINVAL;
    memcpy(c->psi, psi, sizeof(cplx) * c->n);
    c->have_psi = 1; c->stale = 1;
    return WDMO_OK;
}

/* x <- x - L floor((x + L/2)/L): into [-L/2, L/2)  (reading G16) */
static double wrap_pos(double x, double L)
{
    double y = x - L * floor((x + 0.5 * L) / L);
    if (y >= 0.5 * L) y -= L;       /* guard the rounding case x + L/2 just below a multiple of L */
    if (y < -0.5 * L) y += L;
    return y;
}

int wdmo_set_particles(wdmo_ctx *c, long long np, const double *pos, const double *vel,
                       const double *mass, double mass_scalar)
{
    if (!c || np < 0 || (np > 0 && (!pos || !vel))) return WDMO_EINVAL;
    free(c->pos); free(c->vel); free(c->acc); free(c->mass);
    c->pos = c->vel = c->acc = c->mass = NULL; c->np = 0;
    if (np > 0) {
        c->pos = (double *)malloc(sizeof(double) * 3 * (size_t)np);
        c->vel = (double *)malloc(sizeof(double) * 3 * (size_t)np);
        c->acc = (double *)calloc(3 * (size_t)np, sizeof(double));
        c->mass = (double *)malloc(sizeof(double) * (size_t)np);
        if (!c->pos || !c->vel || !c->acc || !c->mass) return WDMO_ENOMEM;
        for (long long i = 0; i < 3 * np; ++i) { c->pos[i] = wrap_pos(pos[i], c->L); c->vel[i] = vel[i]; }
        for (long long p = 0; p < np; ++p) c->mass[p] = mass ? mass[p] : mass_scalar;
        c->np = np;
    }
    c->stale = 1;
    return WDMO_OK;
}

/* rho = |psi|^2 + CIC(x);  Phi = Poisson(rho);  a = Gather(Phi, x)   (Alg. 1 l.12-15; G8, G22) */
static int update_potential(wdmo_ctx *c)
{
    for (size_t i = 0; i < c->n; ++i) {
        double re = creal(c->psi[i]), im = cimag(c->psi[i]);
        c->rho[i] = re * re + im * im;
    }
    if (c->np > 0) assign_deposit(c, c->rho);
    int rc = poisson(c->rho, c->phi, c->work, c->N, c->L, c->G);
    if (rc) return rc;
    if (c->step_diag_on) memcpy(c->phi_grav, c->phi, c->n * sizeof(double));
    /* Phi_total = Phi_DM + Phi_ext (Alg. 1 l.15); particles feel the total as well (G27) */
    if (c->phi_ext)
        for (size_t i = 0; i < c->n; ++i) c->phi[i] += c->phi_ext[i];
    if (c->np > 0) assign_gather(c);
    return WDMO_OK;
}

static int refresh(wdmo_ctx *c)
{
    if (!c->have_psi) return WDMO_ESTATE;
    if (!c->stale) return WDMO_OK;
    int rc = update_potential(c);
    if (rc) return rc;
    c->stale = 0;
    return WDMO_OK;
}

/* psi *= exp(-i Phi h / mu), h = dt/2  (Eq. 18a/d; N^ = -i Phi) ; v += a h */
static void half_kick(wdmo_ctx *c, double h)
{
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)c->n; ++i) {
        double re = creal(c->psi[i]), im = cimag(c->psi[i]);
        double V = c->phi[i] + c->kappa * (re * re + im * im);      /* Eq. 13-14: V = Phi_total + kappa |psi|^2 */
        double th = -V * h / c->mu;
        c->psi[i] *= cos(th) + I * sin(th);
    }
    /* particle half kick of the FIRST / LAST sub-step (sub-step size dt/nsub, so h/nsub here) */
    if (!c->pstatic)
        for (long long i = 0; i < 3 * c->np; ++i) c->vel[i] += c->acc[i] * (h / c->nsub);
}

/* psi = F^-1{ exp(-i mu k^2 dt/2) F{psi} }  (Eq. 18b) ;  x += v dt, wrapped */
static int drift(wdmo_ctx *c, double dt)
{
    int N = c->N;
    int rc = fft3_inplace(c->psi, N, -1);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int ix = 0; ix < N; ++ix) {
        double kx = wavenumber(ix, N, c->L);
        for (int iy = 0; iy < N; ++iy) {
            double ky = wavenumber(iy, N, c->L);
            for (int iz = 0; iz < N; ++iz) {
                double kz = wavenumber(iz, N, c->L);
                double th = -0.5 * c->mu * (kx * kx + ky * ky + kz * kz) * dt;
                c->psi[((size_t)ix * N + iy) * N + iz] *= cos(th) + I * sin(th);
            }
        }
    }
    rc = fft3_inplace(c->psi, N, +1);
    if (rc) return rc;
    /* particles: nsub drifts of dt/nsub in the potential Phi^n of the start of the step (still in c->phi);
     * between two drifts a full kick (closing + opening half kicks of neighbouring sub-steps) with the
     * acceleration gathered at the new position ("multiple sub-steps within each SPE step") */
    if (!c->pstatic && c->np > 0) {
        double h = dt / c->nsub;
        for (int j = 1; j <= c->nsub; ++j) {
            for (long long i = 0; i < 3 * c->np; ++i) c->pos[i] = wrap_pos(c->pos[i] + c->vel[i] * h, c->L);
            if (j < c->nsub) {
                assign_gather(c);
                for (long long i = 0; i < 3 * c->np; ++i) c->vel[i] += c->acc[i] * h;
            }
        }
    }
    return WDMO_OK;
}

/* one axis of Eq. 22: b(x) = 2 - tanh((x + L/2)/w) + tanh((x - L/2)/w), w = L/nb: 0 inside, -> 1 at the faces */
static double absorb_profile(double x, double L, int nb)
{
    double w = L / (double)nb;
    return 2.0 - tanh((x + 0.5 * L) / w) + tanh((x - 0.5 * L) / w);
}

/* psi *= B(x), B = exp(-alpha (b(x) + b(y) + b(z)) dt)   (Eq. 22; Alg. 1 l.17-18; G28) */
static void absorb(wdmo_ctx *c, double dt)
{
    int N = c->N;
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < N; ++iy)
            for (int iz = 0; iz < N; ++iz) {
                double x = -0.5 * c->L + ix * c->dx, y = -0.5 * c->L + iy * c->dx, z = -0.5 * c->L + iz * c->dx;
                double b = absorb_profile(x, c->L, c->nb) + absorb_profile(y, c->L, c->nb) + absorb_profile(z, c->L, c->nb);
                c->psi[((size_t)ix * N + iy) * N + iz] *= exp(-c->alpha * b * dt);
            }
}

/* order 2: cloud-in-cell (G12, G13); order 3: triangular-shaped cloud (G30).  The potential becomes stale. */
int wdmo_set_assignment(wdmo_ctx *c, int order)
{
    if (!c || (order != 2 && order != 3)) return WDMO_EINVAL;
    c->order = order;
    c->stale = 1;
    return WDMO_OK;
}

/* nsub >= 1 leapfrog sub-steps per SPE step; pstatic != 0: particles are a fixed mass distribution */
int wdmo_set_particle_mode(wdmo_ctx *c, int nsub, int pstatic)
{
    if (!c || nsub < 1) return WDMO_EINVAL;
    c->nsub = nsub;
    c->pstatic = pstatic != 0;
    return WDMO_OK;
}

/* kappa: self-interaction strength; phi_ext: N^3 values or NULL; alpha = 0 switches the absorbing layer off */
int wdmo_set_kick_terms(wdmo_ctx *c, double kappa, const double *phi_ext, double alpha, int nb)
{
    if (!c || alpha < 0 || (alpha > 0 && nb < 1)) return WDMO_EINVAL;
    c->kappa = kappa;
    c->alpha = alpha;
    c->nb = nb;
    free(c->phi_ext);
    c->phi_ext = NULL;
    if (phi_ext) {
        c->phi_ext = (double *)malloc(c->n * sizeof(double));
        if (!c->phi_ext) return WDMO_ENOMEM;
        memcpy(c->phi_ext, phi_ext, c->n * sizeof(double));
    }
    c->stale = 1;
    return WDMO_OK;
}

/* Spectral kinetic energy of the field in c->psi, per axis (Sect. 2.3: the kinetic term of Eq. 1 is
 * -(mu^2/2) psi* lap psi per unit m; in Fourier space lap -> -k^2, pseudo-spectral as in Eq. 18(b)):
 *   T_a = (mu^2/2) sum_k k_a^2 |psi~_k|^2 dV / N^3,   psi~ = DFT3(psi) unnormalised (Parseval: sum_x |psi|^2 = sum_k |psi~|^2 / N^3)
 * T = T_x + T_y + T_z equals K + Q of wdmo_diagnostics in the continuum limit (Eq. 11-12).
 * Uses c->work as scratch (free outside poisson()). */
static int spectral_kinetic(wdmo_ctx *c, double T[3])
{
    int N = c->N;
    memcpy(c->work, c->psi, sizeof(cplx) * c->n);
    int rc = fft3_inplace(c->work, N, -1);
    if (rc) return rc;
    double t[3] = {0, 0, 0};
    for (int ix = 0; ix < N; ++ix) {
        double kx = wavenumber(ix, N, c->L);
        for (int iy = 0; iy < N; ++iy) {
            double ky = wavenumber(iy, N, c->L);
            for (int iz = 0; iz < N; ++iz) {
                double kz = wavenumber(iz, N, c->L);
                cplx v = c->work[((size_t)ix * N + iy) * N + iz];
                double a2 = creal(v) * creal(v) + cimag(v) * cimag(v);
                t[0] += kx * kx * a2; t[1] += ky * ky * a2; t[2] += kz * kz * a2;
            }
        }
    }
    double f = 0.5 * c->mu * c->mu * c->dx * c->dx * c->dx / ((double)N * N * N);
    for (int a = 0; a < 3; ++a) T[a] = f * t[a];
    return WDMO_OK;
}

/* Diagnostics of the state between steps (c) and (d) of Eq. 18: psi_2 (after the drift, before the
 * closing half kick), the source rho = |psi_2|^2 + particles and the potential just solved from it.  These are the
 * quantities a fused GPU step has in hand without another pass over the grid:
 *   [0] M = sum |psi_2|^2 dV      [1] max |psi_2|^2      [2] max |Phi_total|   (Eq. 26 PAPER.md:364-368 needs both maxima)
 *   [3] T = T_x + T_y + T_z of psi_2 (spectral; the drift multiplies psi~ by unit-modulus factors, so T is the same
 *       before and after step (b))     [4] W = 1/2 sum rho Phi_grav dV, rho the whole Poisson source, Phi_grav the
 *       Poisson potential of Eq. 23 (without Phi_ext)     [5..7] T_x, T_y, T_z
 * E = T + W is the conserved energy of the pure SPE (the 1/2 in W is what makes it conserved, P6). */
static int record_step_diag(wdmo_ctx *c)
{
    double T[3], M = 0, W = 0, maxrho = 0, maxphi = 0, dV = c->dx * c->dx * c->dx;
    int rc = spectral_kinetic(c, T);
    if (rc) return rc;
    for (size_t i = 0; i < c->n; ++i) {
        double re = creal(c->psi[i]), im = cimag(c->psi[i]), r = re * re + im * im;
        M += r;
        if (r > maxrho) maxrho = r;
        if (fabs(c->phi[i]) > maxphi) maxphi = fabs(c->phi[i]);
        W += 0.5 * c->rho[i] * c->phi_grav[i];
    }
    c->step_diag[0] = M * dV; c->step_diag[1] = maxrho; c->step_diag[2] = maxphi;
    c->step_diag[3] = T[0] + T[1] + T[2]; c->step_diag[4] = W * dV;
    c->step_diag[5] = T[0]; c->step_diag[6] = T[1]; c->step_diag[7] = T[2];
    c->step_diag_valid = 1;
    return WDMO_OK;
}

int wdmo_set_step_diagnostics(wdmo_ctx *c, int on)
{
    if (!c) return WDMO_EINVAL;
    c->step_diag_on = on != 0;
    c->step_diag_valid = 0;
    if (on && !c->phi_grav) {
        c->phi_grav = (double *)malloc(c->n * sizeof(double));
        if (!c->phi_grav) return WDMO_ENOMEM;
    }
    return WDMO_OK;
}

/* WDMO_ESTATE until a step has run with the recording switched on */
int wdmo_step_diagnostics(wdmo_ctx *c, double *out)
{
    if (!c || !out) return WDMO_EINVAL;
    if (!c->step_diag_valid) return WDMO_ESTATE;
    memcpy(out, c->step_diag, sizeof c->step_diag);
    return WDMO_OK;
}

int wdmo_step(wdmo_ctx *c, int nsteps, double dt)
{
    if (!c || nsteps < 0) return WDMO_EINVAL;
    int rc = refresh(c);
    if (rc) return rc;
    for (int s = 0; s < nsteps; ++s) {
        half_kick(c, 0.5 * dt);                 /* (a) + particle half kick with a^n        */
        rc = drift(c, dt);                      /* (b) + particle drift                      */
        if (rc) return rc;
        rc = update_potential(c);               /* (c) rho, Phi^{n+1}, a^{n+1}               */
        if (rc) return rc;
        if (c->step_diag_on && s == nsteps - 1 && (rc = record_step_diag(c))) return rc;
        half_kick(c, 0.5 * dt);                 /* (d) with the new Phi + closing half kick  */
        if (c->alpha > 0) absorb(c, dt);        /* Alg. 1 l.17-18                            */
    }
    return WDMO_OK;
}

int wdmo_get_psi(wdmo_ctx *c, double *out)
{
    if (!c || !out) return WDMO_EINVAL;
    if (!c->have_psi) return WDMO_ESTATE;
    memcpy(out, c->psi, sizeof(cplx) * c->n);
    return WDMO_OK;
}

int wdmo_get_density(wdmo_ctx *c, double *out)
{
    if (!c || !out) return WDMO_EINVAL;
    int rc = refresh(c);
    if (rc) return rc;
    /* |psi|^2 of the psi that wdmo_get_psi returns, plus the particles (reading G22).  Without an absorbing layer this
     * is the source of the last Poisson solve (a kick leaves |psi| unchanged); with one (Alg. 1 l.17-18 masks psi AFTER
     * the potential of l.13 was solved) it is the density of the attenuated field, while Phi stays the one of l.13. */
    for (size_t i = 0; i < c->n; ++i) {
        double re = creal(c->psi[i]), im = cimag(c->psi[i]);
        out[i] = re * re + im * im;
    }
    if (c->np > 0) assign_deposit(c, out);
    return WDMO_OK;
}

int wdmo_get_potential(wdmo_ctx *c, double *out)
{
    if (!c || !out) return WDMO_EINVAL;
    int rc = refresh(c);
    if (rc) return rc;
    memcpy(out, c->phi, sizeof(double) * c->n);
    return WDMO_OK;
}

int wdmo_get_particles(wdmo_ctx *c, double *pos, double *vel)
{
    if (!c) return WDMO_EINVAL;
    if (pos) memcpy(pos, c->pos, sizeof(double) * 3 * (size_t)c->np);
    if (vel) memcpy(vel, c->vel, sizeof(double) * 3 * (size_t)c->np);
    return WDMO_OK;
}

int wdmo_get_accel(wdmo_ctx *c, double *acc)
{
    if (!c || !acc) return WDMO_EINVAL;
    int rc = refresh(c);
    if (rc) return rc;
    memcpy(acc, c->acc, sizeof(double) * 3 * (size_t)c->np);
    return WDMO_OK;
}

/* Volume-integrated diagnostics of the current state (Sect. 3.5-3.6), gradients by the
 * second-order central differences of Eq. 21, periodic:
 *   out[0] M     = sum |psi|^2 dx^3
 *   out[1] max |psi|^2            out[2] max |Phi_total|           (the maxima of Eq. 26)
 *   out[3] V     = sum rho Phi dx^3                                 (as printed: no 1/2)
 *   out[4] K     = 1/2 sum |rho v|^2 / rho dx^3,  rho v = mu Im(psi* grad psi)   (v = mu grad theta)
 *   out[5] Q     = mu^2/2 sum |grad sqrt(rho)|^2 dx^3              (Eq. 12 with its hbar^2/2m prefactor, per unit m)
 *   out[6] dt_max of Eq. 26 without the safety factor:
 *          0.5 min{ 4/(3 pi) dx^2/mu, 2 pi mu / max|Phi|, 2 pi mu / (|kappa| max|psi|^2) }
 *   out[7] T     = mu^2/2 sum_k k^2 |psi~_k|^2 dx^3 / N^3          (spectral kinetic energy; = K + Q in the continuum)
 *   out[8] W     = 1/2 sum rho Phi dx^3 = V/2                      (the 1/2 that makes E conserved, reading G31)
 *   out[9] E     = T + W                                           (conserved by the pure SPE)
 *   out[10], out[11] reserved (0)
 * Which virial identity the numbers satisfy: the paper prints 2K + 2Q + V = 0 with Q = int |grad sqrt(rho)|^2 and
 * V = int rho Phi; with the hbar^2/2m of Eq. 12 kept in Q and the self-energy counted once
 * (W = V/2) the stationary-state identity of the SPE reads 2 (K + Q) + W = 2 T + W = 0 for the returned K, Q, W
 * (reading G31 in DESIGN.md).
 * Phi is refreshed first if stale. */
int wdmo_diagnostics(wdmo_ctx *c, double *out)
{
    if (!c || !out) return WDMO_EINVAL;
    int rc = refresh(c);
    if (rc) return rc;
    int N = c->N;
    double dx = c->dx, dV = dx * dx * dx, mu = c->mu;
    double M = 0, V = 0, K = 0, Q = 0, maxrho = 0, maxphi = 0;
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < N; ++iy)
            for (int iz = 0; iz < N; ++iz) {
                size_t i = ((size_t)ix * N + iy) * N + iz;
                size_t nb[3][2] = {{((size_t)wrap_index(ix + 1, N) * N + iy) * N + iz, ((size_t)wrap_index(ix - 1, N) * N + iy) * N + iz},
                                   {((size_t)ix * N + wrap_index(iy + 1, N)) * N + iz, ((size_t)ix * N + wrap_index(iy - 1, N)) * N + iz},
                                   {((size_t)ix * N + iy) * N + wrap_index(iz + 1, N), ((size_t)ix * N + iy) * N + wrap_index(iz - 1, N)}};
                cplx p = c->psi[i];
                double rho = creal(p) * creal(p) + cimag(p) * cimag(p);
                M += rho;
                V += rho * c->phi[i];
                if (rho > maxrho) maxrho = rho;
                if (fabs(c->phi[i]) > maxphi) maxphi = fabs(c->phi[i]);
                double j2 = 0, g2 = 0;
                for (int a = 0; a < 3; ++a) {
                    cplx grad = (c->psi[nb[a][0]] - c->psi[nb[a][1]]) / (2.0 * dx);
                    double j = mu * cimag(conj(p) * grad);                       /* rho v along axis a */
                    double gs = (cabs(c->psi[nb[a][0]]) - cabs(c->psi[nb[a][1]])) / (2.0 * dx);   /* grad sqrt(rho) */
                    j2 += j * j;
                    g2 += gs * gs;
                }
                if (rho > 0) K += 0.5 * j2 / rho;
                Q += 0.5 * mu * mu * g2;
            }
    out[0] = M * dV; out[1] = maxrho; out[2] = maxphi; out[3] = V * dV; out[4] = K * dV; out[5] = Q * dV;
    double dtm = 4.0 / (3.0 * M_PI) * dx * dx / mu;
    if (maxphi > 0 && 2.0 * M_PI * mu / maxphi < dtm) dtm = 2.0 * M_PI * mu / maxphi;
    if (c->kappa != 0 && maxrho > 0 && 2.0 * M_PI * mu / (fabs(c->kappa) * maxrho) < dtm) dtm = 2.0 * M_PI * mu / (fabs(c->kappa) * maxrho);
    out[6] = 0.5 * dtm;
    double T[3];
    rc = spectral_kinetic(c, T);
    if (rc) return rc;
    out[7] = T[0] + T[1] + T[2];
    out[8] = 0.5 * out[3];
    out[9] = out[7] + out[8];
    out[10] = out[11] = 0;
    return WDMO_OK;
}

int wdmo_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
