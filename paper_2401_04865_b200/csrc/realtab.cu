// realtab.cu -- host construction of the real-space kernel table of realtab.h (eq. 20; its
// derivative, reading A2): Chebyshev interpolation of N(s) and g_N(s) per interval, evaluated in long double,
// converted to monomials in t in [-1, 1].  Also the host-only test hook pce_real_kernel_host().
#include "pce_internal.h"

#include <cmath>

namespace {

struct KParams { long double a, xi, c64; };

// F(u), F'(u) for any real u (erfc of a negative argument is meant literally)
inline void F_dF(const KParams& k, long double u, long double& F, long double& dF)
{
    const long double x = u * k.xi;
    const long double e = expl(-x * x);
    const long double ec = erfcl(x);
    const long double isp = 0.5641895835477562869480794515607726L;  // 1/sqrt(pi)
    F = (2.0L * x * x + 1.0L) * ec - 2.0L * isp * x * e;
    dF = k.xi * (4.0L * x * ec - 4.0L * isp * e);
}

// N(r) and g_N(r) = -N'(r)/r
inline void N_gN(const KParams& k, long double r, long double& N, long double& g)
{
    long double Fp, dFp, Fm, dFm, Fr, dFr;
    F_dF(k, r + 2.0L * k.a, Fp, dFp);
    F_dF(k, r - 2.0L * k.a, Fm, dFm);
    F_dF(k, r, Fr, dFr);
    const long double B = Fp + Fm - 2.0L * Fr, dB = dFp + dFm - 2.0L * dFr;
    N = k.c64 * B / r;
    const long double dN = k.c64 * (dB - B / r) / r;
    g = -dN / r;
}

int key_of(double s) { return rt_hi(s) >> (20 - RT_BITS); }

// monomial coefficients (in t) of the degree-RT_DEG Chebyshev interpolant through the RT_DEG+1 Chebyshev nodes
void cheb_fit(const long double* f, double* out)
{
    constexpr int n = RT_DEG + 1;
    const long double pi = 3.14159265358979323846264338327950288L;
    long double a[n];
    for (int m = 0; m < n; ++m) {
        long double s = 0.0L;
        for (int j = 0; j < n; ++j) s += f[j] * cosl(pi * m * (j + 0.5L) / n);
        a[m] = (m == 0 ? 1.0L : 2.0L) * s / n;
    }
    // T_0 = 1, T_1 = t, T_{m+1} = 2 t T_m - T_{m-1}
    long double Tm1[n] = {0}, Tm[n] = {0}, mono[n] = {0};
    Tm1[0] = 1.0L;
    Tm[1] = 1.0L;
    for (int k = 0; k < n; ++k) mono[k] += a[0] * Tm1[k];
    if (n > 1)
        for (int k = 0; k < n; ++k) mono[k] += a[1] * Tm[k];
    for (int m = 2; m < n; ++m) {
        long double Tn[n] = {0};
        for (int k = 0; k < n; ++k) {
            if (k > 0) Tn[k] += 2.0L * Tm[k - 1];
            Tn[k] -= Tm1[k];
        }
        for (int k = 0; k < n; ++k) { mono[k] += a[m] * Tn[k]; Tm1[k] = Tm[k]; Tm[k] = Tn[k]; }
    }
    for (int k = 0; k < n; ++k) out[k] = (double)mono[k];
}

}  // namespace

// Host table for (a, xi, r_c): intervals from s_lo = 2^floor(log2((a/4)^2)) to beyond r_c^2.
void realtab_build_host(double a, double xi, double rc, std::vector<double>& tab, RealTable& T)
{
    KParams k;
    k.a = a; k.xi = xi;
    k.c64 = 1.0L / (64.0L * 3.14159265358979323846264338327950288L * k.a * k.a * k.xi * k.xi);
    int e = 0;
    std::frexp(a * a / 16.0, &e);               // a^2/16 = m 2^e, m in [0.5, 1)
    const double s_lo = std::ldexp(1.0, e - 1);  // largest power of two <= a^2/16
    T.s_lo = s_lo;
    T.key_lo = key_of(s_lo);
    T.n_int = key_of(rc * rc * (1.0 + 1e-12)) - T.key_lo + 1;
    if (T.n_int < 1) T.n_int = 1;
    tab.assign((size_t)T.n_int * RT_STRIDE, 0.0);
    constexpr int n = RT_DEG + 1;
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < T.n_int; ++i) {
        const int key = T.key_lo + i;
        const long double s0 = rt_from_hi(key << (20 - RT_BITS));
        const long double w = ldexpl(1.0L, (key >> RT_BITS) - 1023 - RT_BITS);
        long double fN[n], fg[n];
        for (int j = 0; j < n; ++j) {
            const long double t = cosl(pi * (j + 0.5L) / n);
            const long double s = s0 + 0.5L * (t + 1.0L) * w;
            N_gN(k, sqrtl(s), fN[j], fg[j]);
        }
        double cN[n], cg[n];
        cheb_fit(fN, cN);
        cheb_fit(fg, cg);
        for (int kk = 0; kk < n; ++kk) {
            tab[(size_t)kk * T.n_int + i] = cN[kk];
            tab[(size_t)(n + kk) * T.n_int + i] = cg[kk];
        }
    }
    T.tab = tab.data();
}

// Generic table of one smooth function f(s), s in [s_lo', s_hi], with the interval scheme of realtab.h, interval-major:
// tab[interval][RT_DEG + 1] monomial coefficients in t.  Used for the shape factor of the Green's function (zfft.cu).
void chebtab_build(double s_lo, double s_hi, long double (*f)(long double, const void*), const void* ctx, std::vector<double>& tab,
                   int& key_lo, int& n_int)
{
    int e = 0;
    std::frexp(s_lo, &e);
    const double lo = std::ldexp(1.0, e - 1);  // largest power of two <= s_lo
    key_lo = key_of(lo);
    n_int = key_of(s_hi * (1.0 + 1e-12)) - key_lo + 1;
    if (n_int < 1) n_int = 1;
    constexpr int n = RT_DEG + 1;
    tab.assign((size_t)n_int * n, 0.0);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < n_int; ++i) {
        const int key = key_lo + i;
        const long double s0 = rt_from_hi(key << (20 - RT_BITS));
        const long double w = ldexpl(1.0L, (key >> RT_BITS) - 1023 - RT_BITS);
        long double fv[n];
        for (int j = 0; j < n; ++j) {
            const long double t = cosl(pi * (j + 0.5L) / n);
            fv[j] = f(s0 + 0.5L * (t + 1.0L) * w, ctx);
        }
        cheb_fit(fv, &tab[(size_t)i * n]);
    }
}

int realtab_upload(pce_ctx* c)
{
    std::vector<double> tab;
    RealTable T;
    realtab_build_host(c->p.a, c->p.xi, c->p.rc, tab, T);
    PCE_CUDA(c, cudaMalloc(&c->rt_dev, tab.size() * sizeof(double)));
    PCE_CUDA(c, cudaMemcpy(c->rt_dev, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice));
    T.tab = c->rt_dev;
    c->rt = T;
    c->bytes += (long long)(tab.size() * sizeof(double));
    return PCE_OK;
}

// Host-only evaluation of the real-space pair kernel exactly as the device evaluates it (table of realtab.h for
// r >= a/4 plus the closed-form Heaviside term; exact formula below) -- for CPU tests of the table; no GPU needed.
extern "C" int pce_real_kernel_host(double a, double xi, double rc, double eps_f, int n, const double* r, double* R, double* dR)
{
    if (!(a > 0) || !(xi > 0) || !(rc > 0) || !(eps_f > 0) || n < 0 || (n > 0 && (!r || !R || !dR))) return PCE_EINVAL;
    std::vector<double> tab;
    RealTable T;
    realtab_build_host(a, xi, rc, tab, T);
    const double inv16pia2 = 1.0 / (16.0 * PCE_PI * a * a);
    for (int i = 0; i < n; ++i) {
        const double ri = r[i], s = ri * ri;
        if (!(ri > 0.0) || s < T.s_lo || !(ri < rc)) { R[i] = dR[i] = NAN; continue; }  // outside the tabulated range
        double N, g;
        rt_eval(T, s, true, N, g);
        double Rv = N, gv = g;
        if (ri < 2.0 * a) {
            const double m = ri - 2.0 * a;
            Rv -= m * m * inv16pia2 / ri;                                       // Heaviside term of eq. 20 (reading G3)
            gv -= (1.0 / (4.0 * PCE_PI * s) - inv16pia2) / ri;                   // -d/dr of it, over r
        }
        R[i] = Rv / eps_f;
        dR[i] = -gv * ri / eps_f;
    }
    return PCE_OK;
}
