// realtab.h -- piecewise-polynomial table of the smooth part of the real-space kernel (eq. 20).
//
// With F(u) = (2 xi^2 u^2 + 1) erfc(u xi) - (2 xi/sqrt(pi)) u exp(-u^2 xi^2) taken literally for negative u, the six
// exp/erfc terms of eq. 20 are
//     N(r) = [F(r+2a) + F(r-2a) - 2 F(r)] / (64 pi a^2 xi^2 r),
// smooth for all r > 0, and  R(r) = N(r) - H(2a-r) (r-2a)^2/(16 pi a^2 r)  (the Heaviside term, reading G3).
// The table stores, per interval of s = r^2, degree-7 polynomials of N and of g_N = -N'(r)/r (the field kernel:
// E_a -= grad R = g (x_a - x_b)).  Intervals follow the floating-point format of s: RT_SUB per octave (the top
// RT_BITS mantissa bits), so the relative width is constant, no sqrt and no division is needed for r >= 2a, and the
// index is two integer instructions.  Below s_lo (r < a/4: only deeply overlapping shells) the exact formula is used.
#pragma once

constexpr int RT_BITS = 4;               // mantissa bits in the interval key
constexpr int RT_SUB = 1 << RT_BITS;     // intervals per octave of s
constexpr int RT_DEG = 7;                // polynomial degree
constexpr int RT_STRIDE = 2 * (RT_DEG + 1);  // doubles per interval: N coefficients, then g_N coefficients

struct RealTable {
    // [RT_STRIDE][n_int], coefficient-major: lanes that look up different intervals touch consecutive words, so a
    // copy in shared memory is read with few bank conflicts.  Rows 0..RT_DEG: N; rows RT_DEG+1..: g_N.
    const double* tab = nullptr;  // device pointer (global or shared) in kernels, host pointer in the test hook
    int key_lo = 0, n_int = 0;    // key(s) = hi32(s) >> (20 - RT_BITS); interval = key - key_lo
    double s_lo = 0.0;            // first tabulated s
};

#ifdef __CUDACC__
#define RT_HD __host__ __device__ __forceinline__
#else
#define RT_HD inline
#endif

RT_HD int rt_hi(double s)
{
#ifdef __CUDA_ARCH__
    return __double2hiint(s);
#else
    union { double d; unsigned long long u; } v; v.d = s; return (int)(v.u >> 32);
#endif
}

RT_HD double rt_from_hi(int hi)
{
#ifdef __CUDA_ARCH__
    return __hiloint2double(hi, 0);
#else
    union { double d; unsigned long long u; } v; v.u = ((unsigned long long)(unsigned)hi) << 32; return v.d;
#endif
}

// N(s) and g_N(s) from the table; requires s_lo <= s < the table's upper end
RT_HD void rt_eval(const RealTable& T, double s, bool field, double& N, double& g)
{
    const int hi = rt_hi(s);
    const int key = hi >> (20 - RT_BITS);
    const double s0 = rt_from_hi(key << (20 - RT_BITS));
    // 2 / width: width = 2^(e - 1023 - RT_BITS) with e = key >> RT_BITS  ->  exponent field 1023 + 1 + RT_BITS - (e - 1023)
    const double two_inv_w = rt_from_hi((2047 + RT_BITS - (key >> RT_BITS)) << 20);
    const double t = (s - s0) * two_inv_w - 1.0;
    const int n = T.n_int;
    const double* c = T.tab + (key - T.key_lo);
    // Estrin's scheme (degree 7): dependency depth 4 instead of 7 -- the hit loop of k_real_cells is latency-bound
    static_assert(RT_DEG == 7, "rt_eval is written for degree 7");
    const double t2 = t * t, t4 = t2 * t2;
    {
        const double p01 = c[1 * n] * t + c[0], p23 = c[3 * n] * t + c[2 * n], p45 = c[5 * n] * t + c[4 * n], p67 = c[7 * n] * t + c[6 * n];
        N = (p67 * t2 + p45) * t4 + (p23 * t2 + p01);
    }
    if (field) {
        const double* d = c + (RT_DEG + 1) * n;
        const double p01 = d[1 * n] * t + d[0], p23 = d[3 * n] * t + d[2 * n], p45 = d[5 * n] * t + d[4 * n], p67 = d[7 * n] * t + d[6 * n];
        g = (p67 * t2 + p45) * t4 + (p23 * t2 + p01);
    }
}

#ifdef __CUDACC__
// The same from a shared-memory copy laid out with a COMPILE-TIME row stride NS (>= n_int): every coefficient sits at a fixed
// offset from the interval's first word, so the 8 (16 with the field) loads are LDS with immediate offsets -- through the
// generic pointer and the run-time stride of rt_eval each load cost two 64-bit adds and a generic LD (38 % of the instructions
// of the direct pass, ncu).
template <int NS>
__device__ __forceinline__ void rt_eval_sh(const double* sh, int key_lo, double s, bool field, double& N, double& g)
{
    const int hi = __double2hiint(s);
    const int key = hi >> (20 - RT_BITS);
    const double s0 = __hiloint2double(key << (20 - RT_BITS), 0);
    const double two_inv_w = __hiloint2double((2047 + RT_BITS - (key >> RT_BITS)) << 20, 0);
    const double t = (s - s0) * two_inv_w - 1.0;
    const double* c = sh + (key - key_lo);
    const double t2 = t * t, t4 = t2 * t2;
    {
        const double p01 = c[1 * NS] * t + c[0], p23 = c[3 * NS] * t + c[2 * NS], p45 = c[5 * NS] * t + c[4 * NS], p67 = c[7 * NS] * t + c[6 * NS];
        N = (p67 * t2 + p45) * t4 + (p23 * t2 + p01);
    }
    if (field) {
        const double* d = c + (RT_DEG + 1) * NS;
        const double p01 = d[1 * NS] * t + d[0], p23 = d[3 * NS] * t + d[2 * NS], p45 = d[5 * NS] * t + d[4 * NS], p67 = d[7 * NS] * t + d[6 * NS];
        g = (p67 * t2 + p45) * t4 + (p23 * t2 + p01);
    }
}
#endif
