// fft_core.h -- radix-8 / 4 / 2 Stockham butterflies shared by the hand-written FFT passes (zfft.cu: z axis fused with the
// Green's function; fftxy.cu: the (x, y) transforms of a mesh plane).  Device code only; no state.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <vector>

namespace fftcore {

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
// multiply by s i  (s = -1: forward, e^{-2 pi i ...})
template <int S> __device__ __forceinline__ double2 cmuli(double2 a) { return (S < 0) ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x); }

// X[k] = sum_n x[n] W^{nk}, W = exp(S 2 pi i / R), natural order in and out
template <int S> __device__ __forceinline__ void dft2(double2* v)
{
    const double2 a = v[0], b = v[1];
    v[0] = cadd(a, b); v[1] = csub(a, b);
}
template <int S> __device__ __forceinline__ void dft4(double2* c)
{
    const double2 t0 = cadd(c[0], c[2]), t1 = csub(c[0], c[2]), t2 = cadd(c[1], c[3]), t3 = cmuli<S>(csub(c[1], c[3]));
    c[0] = cadd(t0, t2); c[2] = csub(t0, t2); c[1] = cadd(t1, t3); c[3] = csub(t1, t3);
}
template <int S> __device__ __forceinline__ void dft8(double2* x)
{
    const double h = 0.70710678118654752440;
    double2 a[4], b[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) { a[n] = cadd(x[n], x[n + 4]); b[n] = csub(x[n], x[n + 4]); }
    // b[n] *= W^n, W = exp(S i pi / 4): W^1 = (1 + S i)/sqrt2, W^2 = S i, W^3 = (-1 + S i)/sqrt2
    b[1] = make_double2(h * (b[1].x - S * b[1].y), h * (b[1].y + S * b[1].x));
    b[2] = cmuli<S>(b[2]);
    b[3] = make_double2(h * (-b[3].x - S * b[3].y), h * (-b[3].y + S * b[3].x));
    dft4<S>(a);
    dft4<S>(b);
#pragma unroll
    for (int m = 0; m < 4; ++m) { x[2 * m] = a[m]; x[2 * m + 1] = b[m]; }
}
template <int R, int S> __device__ __forceinline__ void dftR(double2* v)
{
    if (R == 8) dft8<S>(v);
    else if (R == 4) dft4<S>(v);
    else dft2<S>(v);
}

// N = 8^n8 * rest (rest = 8 counts as one more radix-8 stage)
template <int N> struct Radices {
    static constexpr int rest = (N == 16 || N == 128 || N == 1024) ? 2 : (N == 32 || N == 256) ? 4 : 8;
    static constexpr int n8 = (N == 16 || N == 32 || N == 64) ? (N == 64 ? 2 : 1) : (N == 128 || N == 256 || N == 512) ? (N == 512 ? 3 : 2) : 3;
};


// Twiddles: stage with Ns butterfly groups needs w_k^r, w_k = exp(S 2 pi i k / (Ns R)), k = b mod Ns.  They come from a compact
// table per stage, tws[st] = [w_k | w_k^2 | w_k^4] (k < Ns, forward sign), so that the lanes of a warp read consecutive entries
// (the full-length table indexed by k N / (Ns R) puts them a stride apart: bank conflicts); the rest are products.
template <int R, int S>
__device__ __forceinline__ void twiddle_dft_c(double2* v, const double2* __restrict__ t, int Ns, int k)
{
    if (Ns > 1) {
        double2 w1 = t[k];
        if (S > 0) w1.y = -w1.y;
        if (R == 2) {
            v[1] = cmul(v[1], w1);
        } else {
            double2 w2 = t[Ns + k];
            if (S > 0) w2.y = -w2.y;
            const double2 w3 = cmul(w1, w2);
            v[1] = cmul(v[1], w1);
            v[2] = cmul(v[2], w2);
            v[3] = cmul(v[3], w3);
            if (R == 8) {
                double2 w4 = t[2 * Ns + k];
                if (S > 0) w4.y = -w4.y;
                v[4] = cmul(v[4], w4);
                v[5] = cmul(v[5], cmul(w4, w1));
                v[6] = cmul(v[6], cmul(w4, w2));
                v[7] = cmul(v[7], cmul(w4, w3));
            }
        }
    }
    dftR<R, S>(v);
}

// offset of the table of the stage with Ns groups: stages Ns = 8, 64, 512 hold 3 Ns entries each
__host__ __device__ constexpr int tw_offset(int Ns) { return Ns <= 8 ? 0 : Ns <= 64 ? 24 : Ns <= 512 ? 24 + 192 : 24 + 192 + 1536; }
template <int N> struct TwSize { static constexpr int value = tw_offset(N / Radices<N>::rest) + 3 * (N / Radices<N>::rest); };


// v[r] *= w^r, w = exp(S 2 pi i tstep / N) (table tw[m] = exp(-2 pi i m / N)), then the radix-R butterfly
template <int R, int S>
__device__ __forceinline__ void twiddle_dft(double2* v, int tstep, const double2* __restrict__ tw)
{
    if (tstep != 0) {
        // w, w^2, w^4 from the table (three loads instead of seven: threads of a warp read different k, i.e. conflicting
        // banks), the rest by products
        double2 w1 = tw[tstep];
        if (S > 0) w1.y = -w1.y;
        if (R == 2) {
            v[1] = cmul(v[1], w1);
        } else {
            double2 w2 = tw[2 * tstep];
            if (S > 0) w2.y = -w2.y;
            const double2 w3 = cmul(w1, w2);
            v[1] = cmul(v[1], w1);
            v[2] = cmul(v[2], w2);
            v[3] = cmul(v[3], w3);
            if (R == 8) {
                double2 w4 = tw[4 * tstep];
                if (S > 0) w4.y = -w4.y;
                v[4] = cmul(v[4], w4);
                v[5] = cmul(v[5], cmul(w4, w1));
                v[6] = cmul(v[6], cmul(w4, w2));
                v[7] = cmul(v[7], cmul(w4, w3));
            }
        }
    }
    dftR<R, S>(v);
}

// One Stockham stage of radix R on the thread's 8 elements (8/R butterflies).  in/out: element i of the pencil at
// base[i * stride].  Loads (with the optional per-element scale g, radix 8 only), barrier if in place, stores.
template <int N, int R, int S, bool SYNC>
__device__ __forceinline__ void stage(const double2* in, size_t istr, bool in_ok, double2* out, size_t ostr, bool out_ok, int Ns, int j,
                                      const double2* __restrict__ tw, const double* g)
{
    constexpr int NB = 8 / R;          // butterflies per thread
    constexpr int NT = N / 8;          // threads per pencil
    double2 v[8];
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = j + q * NT;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double2 e = in_ok ? in[(size_t)(b + r * (N / R)) * istr] : make_double2(0.0, 0.0);
            if (g) { e.x *= g[r]; e.y *= g[r]; }
            v[q * R + r] = e;
        }
    }
    if (SYNC) __syncthreads();
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = j + q * NT;
        const int k = b & (Ns - 1);
        twiddle_dft_c<R, S>(v + q * R, tw + tw_offset(Ns), Ns, k);
        const int d = (b - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (out_ok) out[(size_t)(d + r * Ns) * ostr] = v[q * R + r];
    }
}



// host: the per-stage tables of an n-point transform, n = 8^m * rest: stages Ns = 8, 64, ... of radix 8 but for the last one
inline void stage_twiddles(int n, std::vector<double2>& tw)
{
    int rest = n;
    while (rest > 8) rest /= 8;
    const long double pi = 3.14159265358979323846264338327950288L;
    tw.clear();
    for (int Ns = 8; Ns < n; Ns *= 8) {
        const int R = (Ns * 8 <= n) ? 8 : rest;
        tw.resize(tw_offset(Ns));  // no-op by construction of tw_offset
        for (int pw = 1; pw <= 4; pw *= 2)
            for (int k = 0; k < Ns; ++k) {
                const long double ang = -2.0L * pi * (long double)(pw * k) / (long double)(Ns * R);
                tw.push_back(make_double2((double)cosl(ang), (double)sinl(ang)));
            }
    }
    if (tw.empty()) tw.push_back(make_double2(1.0, 0.0));
}

}  // namespace fftcore
