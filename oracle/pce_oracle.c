/*
 * pce_oracle.c -- CPU oracle for the polarizable-colloid electrostatics hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call
 * this file.  It shares no code, header, table or constant with the CUDA
 * path under paper_2401_04865_b200/csrc/ and neither includes the other.
 *
 * What it is: the plain definition of the paper's potential tensor
 *     M_ab = 1/(eps_f V) sum_{k != 0} j0(ka)^2 exp(i k.(x_a - x_b)) / k^2
 * (eq. 9, prefactor read as 1/(eps_f V), reading G2),
 * evaluated to ~1e-14 by a mesh-free direct Ewald sum following the paper's
 * own split, eq. 19: all periodic images inside the oracle's
 * own cut-off in real space (eq. 20; self term eq. 21,
 * PAPER.md:189) plus the structure-factor sum over a half space of wave
 * vectors with h(k) = exp(-k^2/4 xi^2), minus the constant the
 * k = 0 removal leaves behind (reading A1).
 * No mesh, no FFT, no cell list, no blocking: loops over targets, sources,
 * images and wave vectors exactly as the formulas are written.
 *
 * Arithmetic: IEEE double inputs/outputs; the pair kernel and the long sums
 * are carried in x87 long double so that the second-difference cancellation
 * in eq. 20 (terms ~ 1/(64 pi a^2 xi^2 r) cancelling to O(1/r)) does not
 * cost digits.
 *
 * Pins (tests/test_oracle_*.py): eq. 10 vs the quadrature of the shell-shell
 * average; eq. 20/21 vs the radial Fourier integral; d/dr eq. 20 vs finite
 * differences; xi-independence; symmetry / positive definiteness; shell vs
 * textbook point-charge Ewald offset a^2/(3V); the NaCl Madelung constant;
 * a brute-force image sum; solve invariants; conducting-sphere dipole
 * (eq. 33); forces = -grad W by finite differences.
 * Unpinned: the plotted values of the paper's Figs. 1-6 (not printed).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;
#define ORC_PI 3.14159265358979323846264338327950288L

/* ------------------------------------------------------------------ */
/* Pair kernels (eps_f = 1; callers divide by eps_f)                   */
/* ------------------------------------------------------------------ */

/* eq. 10, dimensionally repaired (reading G1):
 * mutual potential of two uniformly charged shells of radius a. */
static ld M_free_ld(ld r, ld a)
{
    if (r >= 2 * a) return 1 / (4 * ORC_PI * r);
    return (4 * a - r) / (16 * ORC_PI * a * a);
}

/* eq. 21: the r -> 0 limit of eq. 20. */
static ld R0_ld(ld a, ld xi)
{
    return (1 - expl(-4 * a * a * xi * xi)) / (8 * ORC_PI * sqrtl(ORC_PI) * a * a * xi)
         + erfcl(2 * a * xi) / (4 * ORC_PI * a);
}

/* eq. 20 term by term, Heaviside sign per reading G3.
 * erfc of the negative argument (r-2a) xi is meant literally. */
static ld R_ld(ld r, ld a, ld xi)
{
    if (r < 1e-6L * a) /* 0/0 region: R(0) + slope of the shell overlap term */
        return R0_ld(a, xi) - r / (16 * ORC_PI * a * a);
    const ld p = r + 2 * a, m = r - 2 * a;
    const ld pi32 = ORC_PI * sqrtl(ORC_PI);
    ld v = 0;
    v += -p / (32 * pi32 * a * a * xi * r) * expl(-p * p * xi * xi);
    v += -m / (32 * pi32 * a * a * xi * r) * expl(-m * m * xi * xi);
    v += 1 / (16 * pi32 * a * a * xi) * expl(-r * r * xi * xi);
    v += (2 * xi * xi * p * p + 1) / (64 * ORC_PI * a * a * xi * xi * r) * erfcl(p * xi);
    v += (2 * xi * xi * m * m + 1) / (64 * ORC_PI * a * a * xi * xi * r) * erfcl(m * xi);
    v += -(2 * xi * xi * r * r + 1) / (32 * ORC_PI * a * a * xi * xi * r) * erfcl(r * xi);
    if (r < 2 * a) v -= 1 / (4 * ORC_PI * r) - (4 * a - r) / (16 * ORC_PI * a * a);
    return v;
}

/* d/dr of eq. 20 -- not printed in the paper (reading A2).
 * With F(u) = (2 xi^2 u^2 + 1) erfc(u xi) - (2 xi/sqrt(pi)) u exp(-u^2 xi^2)
 * the six exp/erfc terms of eq. 20 are  c/r [F(r+2a) + F(r-2a) - 2 F(r)],
 * c = 1/(64 pi a^2 xi^2), and F'(u) = 4 xi^2 u erfc(u xi) - (4 xi/sqrt(pi)) exp(-u^2 xi^2). */
static ld Ffun(ld u, ld xi)
{
    return (2 * xi * xi * u * u + 1) * erfcl(u * xi)
         - (2 * xi / sqrtl(ORC_PI)) * u * expl(-u * u * xi * xi);
}
static ld dFfun(ld u, ld xi)
{
    return 4 * xi * xi * u * erfcl(u * xi) - (4 * xi / sqrtl(ORC_PI)) * expl(-u * u * xi * xi);
}
static ld dR_ld(ld r, ld a, ld xi)
{
    if (r < 1e-6L * a) return -1 / (16 * ORC_PI * a * a);
    const ld p = r + 2 * a, m = r - 2 * a;
    const ld c = 1 / (64 * ORC_PI * a * a * xi * xi);
    ld v = -(c / (r * r)) * (Ffun(p, xi) + Ffun(m, xi) - 2 * Ffun(r, xi))
         + (c / r) * (dFfun(p, xi) + dFfun(m, xi) - 2 * dFfun(r, xi));
    if (r < 2 * a) v += 1 / (4 * ORC_PI * r * r) - 1 / (16 * ORC_PI * a * a);
    return v;
}

double orc_M_free(double r, double a) { return (double)M_free_ld(r, a); }
double orc_R(double r, double a, double xi) { return (double)R_ld(r, a, xi); }
double orc_R0(double a, double xi) { return (double)R0_ld(a, xi); }
double orc_dR(double r, double a, double xi) { return (double)dR_ld(r, a, xi); }

/* wave-space weight g(k) = j0(ka)^2 exp(-k^2/4 xi^2)/k^2  (eq. 19 first line) */
static double gk(double k2, double a, double xi)
{
    double k = sqrt(k2), x = k * a;
    double j0 = (x < 1e-8) ? 1.0 - x * x / 6.0 : sin(x) / x;
    return j0 * j0 * exp(-k2 / (4 * xi * xi)) / k2;
}

static double min_image(double d, double L)
{
    return d - L * floor(d / L + 0.5);
}

/* half space of wave vectors: kx>0, or kx==0&&ky>0, or kx==ky==0&&kz>0 */
typedef struct { int n; int *kx, *ky, *kz; double *g; } klist;

static klist build_klist(const double L[3], double a, double xi, double kmax)
{
    klist K; K.n = 0;
    int mx = (int)floor(kmax * L[0] / (2 * M_PI));
    int my = (int)floor(kmax * L[1] / (2 * M_PI));
    int mz = (int)floor(kmax * L[2] / (2 * M_PI));
    size_t cap = (size_t)(mx + 1) * (2 * my + 1) * (2 * mz + 1);
    K.kx = malloc(cap * sizeof(int)); K.ky = malloc(cap * sizeof(int));
    K.kz = malloc(cap * sizeof(int)); K.g = malloc(cap * sizeof(double));
    for (int ix = 0; ix <= mx; ++ix)
        for (int iy = -my; iy <= my; ++iy)
            for (int iz = -mz; iz <= mz; ++iz) {
                if (ix == 0 && (iy < 0 || (iy == 0 && iz <= 0))) continue;
                double kxv = 2 * M_PI * ix / L[0], kyv = 2 * M_PI * iy / L[1], kzv = 2 * M_PI * iz / L[2];
                double k2 = kxv * kxv + kyv * kyv + kzv * kzv;
                if (k2 > kmax * kmax) continue;
                K.kx[K.n] = ix; K.ky[K.n] = iy; K.kz[K.n] = iz; K.g[K.n] = gk(k2, a, xi);
                ++K.n;
            }
    return K;
}
static void free_klist(klist *K) { free(K->kx); free(K->ky); free(K->kz); free(K->g); }

/* ------------------------------------------------------------------ */
/* Direct Ewald evaluation of psi = M q and E = -grad(M q)             */
/* at the targets tidx[0..Nt) (indices into the source list).          */
/*   xi  : the ORACLE's splitting parameter                            */
/*   s   : r_c = s/xi + 2a, k_max = 2 s xi (exp(-s^2) truncation, eq. 23/28;
 *         eq. 20 decays like erfc((r-2a) xi), hence the 2a)            */
/* Returns 0, or -1 on bad arguments.                                  */
/* ------------------------------------------------------------------ */
int orc_ewald_eval(int N, const double *x, const double *y, const double *z, const double *q,
                   int Nt, const int *tidx, const double L[3], double a, double eps,
                   double xi, double s, int want_field,
                   double *psi, double *Ex, double *Ey, double *Ez)
{
    if (N <= 0 || Nt < 0 || a <= 0 || xi <= 0 || s <= 0 || eps <= 0) return -1;
    const double rc = s / xi + 2 * a, kmax = 2 * s * xi; /* shells: tail ~ erfc((r-2a) xi) */
    const double V = L[0] * L[1] * L[2];
    const int mx = (int)ceil(rc / L[0]), my = (int)ceil(rc / L[1]), mz = (int)ceil(rc / L[2]);

    ld qsum = 0;
    for (int b = 0; b < N; ++b) qsum += q[b];
    const ld cst = qsum / (4 * (ld)xi * xi * V);

    ld *ps = calloc(Nt, sizeof(ld)), *ex = calloc(Nt, sizeof(ld)), *ey = calloc(Nt, sizeof(ld)), *ez = calloc(Nt, sizeof(ld));

    /* ---- real-space images (eq. 19 second line, eq. 20, eq. 21) ---- */
#pragma omp parallel for schedule(dynamic, 4)
    for (int t = 0; t < Nt; ++t) {
        const int al = tidx[t];
        ld sp = 0, sx = 0, sy = 0, sz = 0;
        for (int b = 0; b < N; ++b) {
            if (q[b] == 0.0) continue;
            const double dx0 = min_image(x[al] - x[b], L[0]);
            const double dy0 = min_image(y[al] - y[b], L[1]);
            const double dz0 = min_image(z[al] - z[b], L[2]);
            for (int nx = -mx; nx <= mx; ++nx)
                for (int ny = -my; ny <= my; ++ny)
                    for (int nz = -mz; nz <= mz; ++nz) {
                        const double dx = dx0 + nx * L[0], dy = dy0 + ny * L[1], dz = dz0 + nz * L[2];
                        const double r2 = dx * dx + dy * dy + dz * dz;
                        if (r2 >= rc * rc) continue;
                        if (b == al && nx == 0 && ny == 0 && nz == 0) { /* beta = alpha: eq. 21 */
                            sp += R0_ld(a, xi) * q[b];
                            continue;
                        }
                        const double r = sqrt(r2);
                        if (r == 0.0) { sp += R0_ld(a, xi) * q[b]; continue; } /* reading A9 */
                        sp += R_ld(r, a, xi) * q[b];
                        if (want_field) {
                            const ld f = -dR_ld(r, a, xi) * q[b] / r;
                            sx += f * dx; sy += f * dy; sz += f * dz;
                        }
                    }
        }
        ps[t] = sp; ex[t] = sx; ey[t] = sy; ez[t] = sz;
    }

    /* ---- wave-space sum over a half space (eq. 19 first line) ---- */
    klist K = build_klist(L, a, xi, kmax);
    int kmx = 0, kmy = 0, kmz = 0;
    for (int i = 0; i < K.n; ++i) {
        if (K.kx[i] > kmx) kmx = K.kx[i];
        if (abs(K.ky[i]) > kmy) kmy = abs(K.ky[i]);
        if (abs(K.kz[i]) > kmz) kmz = abs(K.kz[i]);
    }
    /* phase tables cos/sin(2 pi kappa x / L), layout [kappa][particle] */
    double *cxT = malloc((size_t)(kmx + 1) * N * sizeof(double)), *sxT = malloc((size_t)(kmx + 1) * N * sizeof(double));
    double *cyT = malloc((size_t)(kmy + 1) * N * sizeof(double)), *syT = malloc((size_t)(kmy + 1) * N * sizeof(double));
    double *czT = malloc((size_t)(kmz + 1) * N * sizeof(double)), *szT = malloc((size_t)(kmz + 1) * N * sizeof(double));
#pragma omp parallel for schedule(static)
    for (int b = 0; b < N; ++b) {
        for (int k = 0; k <= kmx; ++k) { double ph = 2 * M_PI * k * (x[b] / L[0]); cxT[(size_t)k * N + b] = cos(ph); sxT[(size_t)k * N + b] = sin(ph); }
        for (int k = 0; k <= kmy; ++k) { double ph = 2 * M_PI * k * (y[b] / L[1]); cyT[(size_t)k * N + b] = cos(ph); syT[(size_t)k * N + b] = sin(ph); }
        for (int k = 0; k <= kmz; ++k) { double ph = 2 * M_PI * k * (z[b] / L[2]); czT[(size_t)k * N + b] = cos(ph); szT[(size_t)k * N + b] = sin(ph); }
    }
    /* S(k) = sum_b q_b exp(-i k.x_b) */
    double *Sre = malloc((size_t)K.n * sizeof(double)), *Sim = malloc((size_t)K.n * sizeof(double));
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < K.n; ++i) {
        const int ax = K.kx[i], ay = abs(K.ky[i]), az = abs(K.kz[i]);
        const double sgy = K.ky[i] < 0 ? -1.0 : 1.0, sgz = K.kz[i] < 0 ? -1.0 : 1.0;
        const double *cx = cxT + (size_t)ax * N, *sx = sxT + (size_t)ax * N;
        const double *cy = cyT + (size_t)ay * N, *sy = syT + (size_t)ay * N;
        const double *cz = czT + (size_t)az * N, *sz = szT + (size_t)az * N;
        ld re = 0, im = 0;
        for (int b = 0; b < N; ++b) {
            /* e^{i k.x} = (cx+i sx)(cy+i sgy sy)(cz+i sgz sz) */
            const double c1 = cx[b] * cy[b] - sx[b] * sgy * sy[b];
            const double s1 = sx[b] * cy[b] + cx[b] * sgy * sy[b];
            const double c2 = c1 * cz[b] - s1 * sgz * sz[b];
            const double s2 = s1 * cz[b] + c1 * sgz * sz[b];
            re += q[b] * c2; im -= q[b] * s2;
        }
        Sre[i] = (double)re; Sim[i] = (double)im;
    }
#pragma omp parallel for schedule(dynamic, 4)
    for (int t = 0; t < Nt; ++t) {
        const int al = tidx[t];
        ld sp = 0, sx_ = 0, sy_ = 0, sz_ = 0;
        for (int i = 0; i < K.n; ++i) {
            const int ax = K.kx[i], ay = abs(K.ky[i]), az = abs(K.kz[i]);
            const double sgy = K.ky[i] < 0 ? -1.0 : 1.0, sgz = K.kz[i] < 0 ? -1.0 : 1.0;
            const double cxa = cxT[(size_t)ax * N + al], sxa = sxT[(size_t)ax * N + al];
            const double cya = cyT[(size_t)ay * N + al], sya = sgy * syT[(size_t)ay * N + al];
            const double cza = czT[(size_t)az * N + al], sza = sgz * szT[(size_t)az * N + al];
            const double c1 = cxa * cya - sxa * sya, s1 = sxa * cya + cxa * sya;
            const double c2 = c1 * cza - s1 * sza, s2 = s1 * cza + c1 * sza;
            /* S e^{ik.x}: Re = Sre c2 - Sim s2 ; Im = Sre s2 + Sim c2 */
            const double re = Sre[i] * c2 - Sim[i] * s2;
            sp += K.g[i] * re;
            if (want_field) {
                const double im = Sre[i] * s2 + Sim[i] * c2;
                const double w = K.g[i] * im;
                sx_ += w * (2 * M_PI * K.kx[i] / L[0]);
                sy_ += w * (2 * M_PI * K.ky[i] / L[1]);
                sz_ += w * (2 * M_PI * K.kz[i] / L[2]);
            }
        }
        ps[t] += 2 * sp / V; ex[t] += 2 * sx_ / V; ey[t] += 2 * sy_ / V; ez[t] += 2 * sz_ / V;
    }
    free(cxT); free(sxT); free(cyT); free(syT); free(czT); free(szT); free(Sre); free(Sim);
    free_klist(&K);

    for (int t = 0; t < Nt; ++t) {
        psi[t] = (double)((ps[t] - cst) / eps);
        if (want_field) { Ex[t] = (double)(ex[t] / eps); Ey[t] = (double)(ey[t] / eps); Ez[t] = (double)(ez[t] / eps); }
    }
    free(ps); free(ex); free(ey); free(ez);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Dense potential tensor M (N x N, row major), entry by entry from    */
/* the pair function  sum_n R(|d+n|) + (2/V) sum_k g cos(k.d) - 1/(4 xi^2 V). */
/* ------------------------------------------------------------------ */
int orc_pair_matrix(int N, const double *x, const double *y, const double *z,
                    const double L[3], double a, double eps, double xi, double s, double *M)
{
    if (N <= 0 || a <= 0 || xi <= 0 || s <= 0 || eps <= 0) return -1;
    const double rc = s / xi + 2 * a, kmax = 2 * s * xi; /* shells: tail ~ erfc((r-2a) xi) */
    const double V = L[0] * L[1] * L[2];
    const int mx = (int)ceil(rc / L[0]), my = (int)ceil(rc / L[1]), mz = (int)ceil(rc / L[2]);
    klist K = build_klist(L, a, xi, kmax);
    const ld cst = 1 / (4 * (ld)xi * xi * V);

#pragma omp parallel for schedule(dynamic, 1)
    for (int al = 0; al < N; ++al) {
        for (int b = al; b < N; ++b) {
            const double dx0 = min_image(x[al] - x[b], L[0]);
            const double dy0 = min_image(y[al] - y[b], L[1]);
            const double dz0 = min_image(z[al] - z[b], L[2]);
            ld v = 0;
            for (int nx = -mx; nx <= mx; ++nx)
                for (int ny = -my; ny <= my; ++ny)
                    for (int nz = -mz; nz <= mz; ++nz) {
                        const double dx = dx0 + nx * L[0], dy = dy0 + ny * L[1], dz = dz0 + nz * L[2];
                        const double r2 = dx * dx + dy * dy + dz * dz;
                        if (r2 >= rc * rc) continue;
                        if ((b == al && nx == 0 && ny == 0 && nz == 0) || r2 == 0.0) v += R0_ld(a, xi);
                        else v += R_ld(sqrt(r2), a, xi);
                    }
            ld kw = 0;
            for (int i = 0; i < K.n; ++i) {
                const double ph = 2 * M_PI * (K.kx[i] * (dx0 / L[0]) + K.ky[i] * (dy0 / L[1]) + K.kz[i] * (dz0 / L[2]));
                kw += K.g[i] * cos(ph);
            }
            v += 2 * kw / V - cst;
            M[(size_t)al * N + b] = M[(size_t)b * N + al] = (double)(v / eps);
        }
    }
    free_klist(&K);
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
