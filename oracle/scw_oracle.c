/*
 * scw_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the sCWatter field-evaluation hot
 * path computes (arxiv 2404.07293; citations are PAPER.md line numbers).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may build, load or call this file.  It shares no code,
 * header, table or helper with paper_2404_07293_b200/csrc (the CUDA path).
 *
 * What is evaluated is the plain definition: the discrete form of eq. 3
 * (PAPER.md:50-55),
 *
 *     E(r) = sum_j sum_m  p_{m,j} * exp[ i k ( s_{m,j} . (r - r_ref,j) ) ],
 *
 * one term at a time, in the paper's order and notation, with no factoring,
 * blocking or re-association beyond what is stated next to each function.
 * Accumulation is in long double so the oracle is the more accurate side.
 *
 * Pins (tests/test_oracle_pins.py): eq. 2 special cases, eq. 6 index map,
 * eq. 7 semigroup, |w|<=1 reference-plane invariant, single-mode closed
 * form, ifft2 on commensurate grids, Parseval, periodicity, homogeneous-layer
 * TE/TM plane waves with s.p=0 (eq. 14), brute-force DFT on 3x3 toys; the dir == NULL branch (scwo_dir) against the
 * hand-derived table tests/golden/dir_cases.txt through the single-mode closed form.
 * Parity unpinned: the statistical content of the synthetic V, c, gamma
 * (synthetic by construction) -- see DESIGN.md.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SCWO_PI 3.14159265358979323846264338327950288

/* Number of threads the sample loops will use (reported as `cores`). */
int scwo_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void scwo_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/*
 * eq. 2: s_z = sqrt(n^2 - sx^2 - sy^2), with the branch the
 * paper leaves open read as Im >= 0 (and Re >= 0 when Im == 0)
 * [DESIGN.md reading c-2].  out[0]=Re, out[1]=Im.
 */
void scwo_sz(double n_re, double n_im, double sx, double sy, double *out)
{
    double complex n = n_re + n_im * I;
    double complex a = n * n - (sx * sx + sy * sy);
    /* guard the -0.0 imaginary part: csqrt(-x - 0i) = -i sqrt(x) in C */
    if (cimag(a) == 0.0) a = creal(a) + 0.0 * I;
    double complex g = csqrt(a);
    if (cimag(g) < 0.0 || (cimag(g) == 0.0 && creal(g) < 0.0)) g = -g;
    out[0] = creal(g);
    out[1] = cimag(g);
}

/*
 * eq. 6 index map: m -> (u, v) with
 * v = floor(m/U) - floor(V/2), u = (m mod U) - floor(U/2) [reading c-5].
 */
void scwo_index_map(int U, int Vn, int m, int *u, int *v)
{
    *v = m / U - Vn / 2;
    *u = m % U - U / 2;
}

/*
 * eq. 7: G(A, z_a, z_b) = exp[ i k (z_b - z_a) A ],
 * k = 2 pi / lambda, A complex.  Written as modulus * unit phasor; the phase
 * in turns is reduced with remainder(), which is exact in fp64.
 */
static double complex scwo_G(double complex A, double za, double zb, double lambda)
{
    double dz = zb - za;
    double amp = exp(-2.0 * SCWO_PI * cimag(A) * dz / lambda);
    double t = remainder(creal(A) * dz / lambda, 1.0);
    return amp * (cos(2.0 * SCWO_PI * t) + I * sin(2.0 * SCWO_PI * t));
}

void scwo_green(double A_re, double A_im, double za, double zb, double lambda, double *out)
{
    double complex g = scwo_G(A_re + A_im * I, za, zb, lambda);
    out[0] = creal(g);
    out[1] = cimag(g);
}

/* dir[j] given, or derived from the sign of gamma_j when dir == NULL:
 * a "+" mode has gamma = +sqrt(...) (Im >= 0), a "-" mode gamma = -sqrt(...). */
static int scwo_dir(const int8_t *dir, const double complex *gamma, int64_t j)
{
    if (dir) return dir[j] > 0 ? 1 : -1;
    double gi = cimag(gamma[j]), gr = creal(gamma[j]);
    return (gi > 0.0 || (gi == 0.0 && gr >= 0.0)) ? 1 : -1;
}

static double complex scwo_loadV(const void *V, int v_is_f32, int64_t idx)
{
    if (v_is_f32) {
        const float *p = (const float *)V + 2 * idx;
        return (double)p[0] + (double)p[1] * I;
    }
    const double *p = (const double *)V + 2 * idx;
    return p[0] + p[1] * I;
}

/*
 * Tier A -- interior field of one layer at n arbitrary samples.
 * eq. 34 read as eq. 10 applied to eq. 31 (
 * reading c-4), with eq. 30's reference planes:
 *
 *   E_comp(x,y,z) = sum_j sum_m  c_j V[comp*M+m, j]
 *                     * exp(i k s_m.(x,y)) * G(gamma_j, zref_j, z)
 *   zref_j = z_lo (= z_{l-1}) for "+" modes, z_hi (= z_l) for "-" modes,
 *   k s_m.(x,y) = 2 pi (u x / X + v y / Y)                  (eq. 6, eq. 10).
 *
 * Plain sum: no 1/M factor (eq. 10 as printed; reading c-6).
 * V: column-major [ldV x J] complex (interleaved re,im), rows comp*M+m
 * (P = [P_x; P_y; P_z], eq. 28; reading c-8); c may be NULL (= ones).
 * xyz: [n][3] doubles.  E: [n][3] complex128, comp fastest.
 * The only parallelism is over samples (independent sums).
 */
void scwo_layer_samples(int U, int Vn, double X, double Y, double lambda,
                        double z_lo, double z_hi, int64_t J,
                        const void *V, int v_is_f32, int64_t ldV,
                        const double *c, const double *gamma_, const int8_t *dir,
                        int64_t n, const double *xyz, double *E_)
{
    const double complex *gamma = (const double complex *)gamma_;
    const double complex *cc = (const double complex *)c;
    double complex *E = (double complex *)E_;
    const int64_t M = (int64_t)U * Vn;

#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < n; ++s) {
        const double x = xyz[3 * s + 0], y = xyz[3 * s + 1], z = xyz[3 * s + 2];
        long double acc_re[3] = {0.0L, 0.0L, 0.0L}, acc_im[3] = {0.0L, 0.0L, 0.0L};
        for (int64_t j = 0; j < J; ++j) {                        /* modes, eq. 23/31 */
            const double zref = scwo_dir(dir, gamma, j) > 0 ? z_lo : z_hi;
            const double dz = z - zref;
            const double gr = creal(gamma[j]), gi = cimag(gamma[j]);
            const double a = exp(-2.0 * SCWO_PI * gi * dz / lambda);      /* decay <= 1 */
            const double complex cj = cc ? cc[j] : 1.0;
            for (int64_t m = 0; m < M; ++m) {                    /* frequencies, eq. 10 */
                int u, v;
                scwo_index_map(U, Vn, (int)m, &u, &v);
                double t = u * x / X + v * y / Y + gr * dz / lambda;   /* phase in turns */
                t = remainder(t, 1.0);
                const double complex w = a * (cos(2.0 * SCWO_PI * t) + I * sin(2.0 * SCWO_PI * t));
                for (int comp = 0; comp < 3; ++comp) {
                    const double complex term =
                        cj * scwo_loadV(V, v_is_f32, j * ldV + comp * M + m) * w;
                    acc_re[comp] += creal(term);
                    acc_im[comp] += cimag(term);
                }
            }
        }
        for (int comp = 0; comp < 3; ++comp)
            E[3 * s + comp] = (double)acc_re[comp] + (double)acc_im[comp] * I;
    }
}

/*
 * Plane-wave form (eq. 3 / eq. 9-10; PAPER.md:87
 * allows any set of s_m): one plane wave per mode,
 *
 *   E(r) = sum_j p_j exp( i k [ sx_j x + sy_j y + gamma_j (z - zref_j) ] ).
 *
 * sx, sy: [J] doubles (direction cosines, eq. 6: s = lambda (u/X, v/Y)),
 * gamma: [J] complex128, zref: [J], p: [J][3] complex128 (or complex64 when
 * p_is_f32), xyz: [n][3], E: [n][3] complex128.
 */
void scwo_planewaves(int64_t J, double lambda, const double *sx, const double *sy,
                     const double *gamma_, const double *zref,
                     const void *p, int p_is_f32,
                     int64_t n, const double *xyz, double *E_)
{
    const double complex *gamma = (const double complex *)gamma_;
    double complex *E = (double complex *)E_;

#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < n; ++s) {
        const double x = xyz[3 * s + 0], y = xyz[3 * s + 1], z = xyz[3 * s + 2];
        long double acc_re[3] = {0.0L, 0.0L, 0.0L}, acc_im[3] = {0.0L, 0.0L, 0.0L};
        for (int64_t j = 0; j < J; ++j) {
            const double dz = z - zref[j];
            const double a = exp(-2.0 * SCWO_PI * cimag(gamma[j]) * dz / lambda);
            double t = (sx[j] * x + sy[j] * y + creal(gamma[j]) * dz) / lambda;
            t = remainder(t, 1.0);
            const double complex w = a * (cos(2.0 * SCWO_PI * t) + I * sin(2.0 * SCWO_PI * t));
            for (int comp = 0; comp < 3; ++comp) {
                const double complex term = scwo_loadV(p, p_is_f32, 3 * j + comp) * w;
                acc_re[comp] += creal(term);
                acc_im[comp] += cimag(term);
            }
        }
        for (int comp = 0; comp < 3; ++comp)
            E[3 * s + comp] = (double)acc_re[comp] + (double)acc_im[comp] * I;
    }
}
