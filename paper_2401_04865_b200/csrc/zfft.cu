// zfft.cu -- steps 3-5 of the spectral Ewald algorithm with the z axis fused:
//   cuFFT 2-D D2Z per mesh plane (x, y)  ->  k_zfft_scale: FFT along z, multiply by the Green's function of eq. 26
//   (PAPER.md:219), inverse FFT along z, all in shared memory  ->  cuFFT 2-D Z2D per plane.
// The separate passes (cuFFT z pass, k_scale, cuFFT z pass) move the 1.08 GB half spectrum through HBM three times
// (6 x 1.08 GB at 512^3); fused, it is read once and written once.  cuFFT stays the only library call and does the
// (x, y) transforms.  Available for power-of-two N_z in 16..1024; other meshes use the 3-D cuFFT plans + k_scale (wave.cu).
//
// Layout: gk[z][y][kx] complex128.  A CTA owns a tile of KP = 4 consecutive kx of one row y (64 contiguous bytes per z) and then
// the mirror row N_y - y, for which the Green's function values are the same (computed once per CTA into shared memory, the
// Gaussian factor from per-axis host tables).  Thread (j, p): pencil p = kx0 + p, butterfly index j.  Shared tile [z][KP]: the
// pencils of a z are consecutive, so every warp access is conflict-free.
// Stockham autosort, radix 8 (the rest radix 4 or 2), in place with a barrier between the loads and the stores of a stage;
// the first forward stage reads global memory, the last inverse stage writes it.  Twiddles exp(-2 pi i m / N) come from a
// host-computed table.  The z transform pair needs no particular sign convention: the Green's function is even in k_z.
#include "pce_internal.h"
#include "fft_core.h"

#include <cmath>
#include <cstdlib>

namespace {

using namespace fftcore;

// j0(ka)^2 / k^2 at s = k^2 > 0: degree-7 polynomial of the interval of s (intervals follow the floating-point format of s,
// 16 per octave, as in realtab.h; host table in long double, zfft_init)
__device__ __forceinline__ double shape_eval(const double* __restrict__ tab, int key_lo, double s)
{
    const int key = __double2hiint(s) >> (20 - RT_BITS);
    const double s0 = __hiloint2double(key << (20 - RT_BITS), 0);
    const double two_inv_w = __hiloint2double((2047 + RT_BITS - (key >> RT_BITS)) << 20, 0);
    const double t = (s - s0) * two_inv_w - 1.0;
    const double* c = tab + (size_t)(key - key_lo) * (RT_DEG + 1);
    const double2 c01 = __ldg(reinterpret_cast<const double2*>(c)), c23 = __ldg(reinterpret_cast<const double2*>(c + 2));
    const double2 c45 = __ldg(reinterpret_cast<const double2*>(c + 4)), c67 = __ldg(reinterpret_cast<const double2*>(c + 6));
    const double t2 = t * t, t4 = t2 * t2;
    return ((c67.y * t + c67.x) * t2 + (c45.y * t + c45.x)) * t4 + ((c23.y * t + c23.x) * t2 + (c01.y * t + c01.x));
}

// last forward stage x Green's function x first inverse stage on the tile column sp (stride KP), in place
// deriv = 0, 1, 2: additionally multiply by -i k_d (ik differentiation: the field component E_d = -d psi / d x_d in wave
// space); kxy = k_x or k_y of the thread's pencil (0 at the Nyquist mode), kzfac = 2 pi / L_z
template <int N, int R>
__device__ __forceinline__ void fused_middle(double2* sp, int j, int p, const double2* __restrict__ tw, const double* __restrict__ gs,
                                             int deriv, double kxy, double kzfac);


// forward (S = -1): stages 8 (global -> smem), 8.., rest (-> smem);  inverse (S = +1): 8 (smem, scaled -> smem), 8.., rest (-> global)
// KP pencils per CTA, N/8 threads per pencil.  zexp = [ex | ey | ez]: exp(-gexp_d k_d^2) per axis (host tables).
constexpr int KP = 4;
template <int N, int R>
__device__ __forceinline__ void fused_middle(double2* sp, int j, int p, const double2* __restrict__ tw, const double* __restrict__ gs,
                                             int deriv, double kxy, double kzfac)
{
    constexpr int NB = 8 / R, NTH = N / 8;
    double2 v[8];
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = j + q * NTH;
#pragma unroll
        for (int r = 0; r < R; ++r) v[q * R + r] = sp[(size_t)(b + r * (N / R)) * KP];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = j + q * NTH;  // b < N / R = Ns: k = b, twiddle step k N / (Ns R) = b
        twiddle_dft_c<R, -1>(v + q * R, tw + tw_offset(N / R), N / R, b);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int iz = b + r * (N / R);
            const double gf = gs[iz * KP + p];
            v[q * R + r].x *= gf; v[q * R + r].y *= gf;
            if (deriv >= 0) {  // -i k_d (x + i y) = k_d (y - i x); the Nyquist mode has no derivative on an even mesh
                const double kd = (deriv == 2) ? kzfac * (double)(iz < N / 2 ? iz : (iz == N / 2 ? 0 : iz - N)) : kxy;
                v[q * R + r] = make_double2(v[q * R + r].y * kd, -v[q * R + r].x * kd);
            }
        }
    }
    // first inverse stage, radix 8 (the same stage order as the forward transform, so both share the twiddle tables): the
    // thread holds the elements j + m N/8, slot (q, r) of the radix-R stage being m = q + r 8/R
    double2 w[8];
#pragma unroll
    for (int q = 0; q < NB; ++q)
#pragma unroll
        for (int r = 0; r < R; ++r) w[q + r * NB] = v[q * R + r];
    dft8<+1>(w);  // Ns = 1: no twiddles; outputs at 8 j + r
#pragma unroll
    for (int r = 0; r < 8; ++r) sp[(size_t)(8 * j + r) * KP] = w[r];
}
template <int N>
__global__ void __launch_bounds__(N / 8 * KP, (N <= 512) ? 3 : 1)
k_zfft_scale(WaveConst wc, const double2* gin, double2* gout, int deriv, const double2* __restrict__ tw_g, const double* __restrict__ zexp,
             const double* __restrict__ shape, int shape_key_lo, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(16) unsigned char zsm[];
    double2* tile = reinterpret_cast<double2*>(zsm);       // [N][KP]
    double2* tw = tile + (size_t)N * KP;                    // per-stage twiddle tables (fft_core.h)
    double* gs = reinterpret_cast<double*>(tw + TwSize<N>::value);  // [N][KP] Green's function of the CTA's pencils
    constexpr int REST = Radices<N>::rest, N8 = Radices<N>::n8;
    const int tid = threadIdx.x, p = tid % KP, j = tid / KP;
    for (int i = tid; i < TwSize<N>::value; i += N / 8 * KP) tw[i] = tw_g[i];
    const int nxh = wc.Nxh, ny = wc.Ng[1];
    const int kxi = blockIdx.x * KP + p, iy = blockIdx.y;  // iy in [0, ny/2]
    const bool col_ok = kxi < nxh;
    const size_t zstr = (size_t)ny * nxh;
    // Green's function (eq. 26, with all constants folded in) of the CTA's pencils into shared memory.  It is even in k_z and
    // in k_y: N/2 + 1 evaluations per pencil serve both halves of the spectrum and both rows (iy and its mirror N_y - iy).
    {
        const double ky = wc.kfac[1] * iy;
        const double* ez = zexp + nxh + ny / 2 + 1;
        for (int e = tid; e < (N / 2 + 1) * KP; e += N / 8 * KP) {
            const int iz = e / KP, pp = e % KP, kxe = blockIdx.x * KP + pp;
            double f = 0.0;  // k = 0 removed; pencils beyond N_x/2 unused
            if (kxe < nxh) {
                const double kx = wc.kfac[0] * kxe, kz = wc.kfac[2] * (double)iz;
                const double k2 = kx * kx + ky * ky + kz * kz;
                if (k2 > 0.0)  // shape factor j0(ka)^2 / k^2 from its table in k^2 (no sqrt, sin or division here)
                    f = wc.scale_norm * zexp[kxe] * zexp[nxh + iy] * ez[iz] * shape_eval(shape, shape_key_lo, k2);
            }
            gs[iz * KP + pp] = f;
            if (iz > 0 && iz < N / 2) gs[(N - iz) * KP + pp] = f;
        }
    }
    const int my = (iy == 0 || 2 * iy == ny) ? -1 : ny - iy;  // mirror row: same |k_y|
    constexpr int NF8 = (REST == 8) ? N8 - 1 : N8;  // radix-8 stages before the fused one
    for (int pass = 0; pass < 2; ++pass) {
        const int y = pass == 0 ? iy : my;
        if (y < 0) break;
        const double2* cin = gin + (size_t)y * nxh + (col_ok ? kxi : 0);
        double2* col = gout + (size_t)y * nxh + (col_ok ? kxi : 0);
        double2* sp = tile + p;
        double kxy = 0.0;
        if (deriv == 0) kxy = (2 * kxi == wc.Ng[0]) ? 0.0 : wc.kfac[0] * kxi;
        if (deriv == 1) kxy = (2 * iy == ny) ? 0.0 : wc.kfac[1] * (pass == 0 ? iy : -iy);
        __syncthreads();  // twiddles and Green's function stored / previous pass done with the tile
        // ---- forward: the first stage reads global memory; all but the last stage of the transform here
        stage<N, 8, -1, false>(cin, zstr, col_ok, sp, KP, true, 1, j, tw, nullptr);
        __syncthreads();
        int Ns = 8;
        if (NF8 >= 2) { stage<N, 8, -1, true>(sp, KP, true, sp, KP, true, Ns, j, tw, nullptr); __syncthreads(); Ns *= 8; }
        if (NF8 >= 3) { stage<N, 8, -1, true>(sp, KP, true, sp, KP, true, Ns, j, tw, nullptr); __syncthreads(); Ns *= 8; }
        // ---- last forward stage (radix REST, Ns = N / REST) x Green's function x first inverse stage (radix REST, Ns = 1), in
        // registers: the forward stage leaves element b + r N/REST in slot r, which is what the inverse stage reads
        fused_middle<N, REST>(sp, j, p, tw, gs, deriv, kxy, wc.kfac[2]);
        __syncthreads();
        // ---- inverse: the remaining radix-8 stages, then the stage of radix REST straight to global memory
        Ns = 8;
        if (NF8 >= 2) { stage<N, 8, +1, true>(sp, KP, true, sp, KP, true, Ns, j, tw, nullptr); __syncthreads(); Ns *= 8; }
        if (NF8 >= 3) { stage<N, 8, +1, true>(sp, KP, true, sp, KP, true, Ns, j, tw, nullptr); __syncthreads(); Ns *= 8; }
        stage<N, REST, +1, false>(sp, KP, true, col, zstr, col_ok, Ns, j, tw, nullptr);
    }
}

template <int N> int launch(pce_ctx* c, const double2* gin, double2* gout, int deriv)
{
    const size_t smem = (size_t)N * KP * sizeof(double2) + (size_t)TwSize<N>::value * sizeof(double2) + (size_t)N * KP * sizeof(double);
    if (!c->zfft_attr_set && smem > 48 * 1024) {  // the attribute is per device: once per context, not per process
        PCE_CUDA(c, cudaFuncSetAttribute(k_zfft_scale<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->zfft_attr_set = true;
    }
    const dim3 grid(cdiv(c->wk.Nxh, KP), c->wk.Ng[1] / 2 + 1);
    k_zfft_scale<N><<<grid, N / 8 * KP, smem, c->st>>>(c->wk, gin, gout, deriv, c->ztw, c->zexp, c->zshape, c->zshape_key_lo, c->skip_flag);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

}  // namespace

bool zfft_supported(const pce_params& p)
{
    const int n = p.Ng[2];
    return (n == 16 || n == 32 || n == 64 || n == 128 || n == 256 || n == 512 || n == 1024) && p.Ng[1] % 2 == 0;
}

// twiddle table exp(-2 pi i m / N_z) (host, long double) and the two batched 2-D cuFFT plans
int zfft_init(pce_ctx* c)
{
    const int n = c->p.Ng[2];
    std::vector<double2> tw;
    stage_twiddles(n, tw);
    PCE_CUDA(c, cudaMalloc(&c->ztw, tw.size() * sizeof(double2)));
    PCE_CUDA(c, cudaMemcpy(c->ztw, tw.data(), tw.size() * sizeof(double2), cudaMemcpyHostToDevice));
    // per-axis factors exp(-(1 - eta_d) k_d^2 / 4 xi^2) of eq. 26: [kx = 0..Nx/2 | ky = 0..Ny/2 | kz = 0..Nz/2], one set per window
    // (eta depends on P, eq. 31)
    const int cnt[3] = {c->wk.Nxh, c->p.Ng[1] / 2 + 1, n / 2 + 1};
    for (int s = 0; s < 2; ++s) {
        std::vector<double> ze;
        for (int d = 0; d < 3; ++d)
            for (int i = 0; i < cnt[d]; ++i) {
                const double k = c->wset[s].kfac[d] * i;
                ze.push_back(std::exp(-c->wset[s].gexp[d] * k * k));
            }
        PCE_CUDA(c, cudaMalloc(&c->zexp_set[s], ze.size() * sizeof(double)));
        PCE_CUDA(c, cudaMemcpy(c->zexp_set[s], ze.data(), ze.size() * sizeof(double), cudaMemcpyHostToDevice));
    }
    c->zexp = c->zexp_set[0];
    // shape factor j0(ka)^2 / k^2 (eq. 9 / eq. 26) as a function of s = k^2 between the smallest and the largest mesh wavenumber
    double smin = 1e300, smax = 0.0;
    for (int d = 0; d < 3; ++d) {
        const double k1 = c->wk.kfac[d], kn = c->wk.kfac[d] * (c->p.Ng[d] / 2);
        smin = std::fmin(smin, k1 * k1);
        smax += kn * kn;
    }
    const long double a = c->p.a;
    std::vector<double> st;
    chebtab_build(smin, smax, [](long double s, const void* ctx) -> long double {
        const long double x = *static_cast<const long double*>(ctx) * sqrtl(s);
        const long double j0 = (x < 1e-6L) ? 1.0L - x * x / 6.0L : sinl(x) / x;
        return j0 * j0 / s;
    }, &a, st, c->zshape_key_lo, c->zshape_n);
    PCE_CUDA(c, cudaMalloc(&c->zshape, st.size() * sizeof(double)));
    PCE_CUDA(c, cudaMemcpy(c->zshape, st.data(), st.size() * sizeof(double), cudaMemcpyHostToDevice));
    return PCE_OK;
}

int zfft_scale(pce_ctx* c, const void* in, void* out, int deriv)
{
    const double2* gin = static_cast<const double2*>(in);
    double2* gout = static_cast<double2*>(out);
    switch (c->p.Ng[2]) {
        case 16: return launch<16>(c, gin, gout, deriv);
        case 32: return launch<32>(c, gin, gout, deriv);
        case 64: return launch<64>(c, gin, gout, deriv);
        case 128: return launch<128>(c, gin, gout, deriv);
        case 256: return launch<256>(c, gin, gout, deriv);
        case 512: return launch<512>(c, gin, gout, deriv);
        case 1024: return launch<1024>(c, gin, gout, deriv);
        default: c->err = "zfft_scale: unsupported N_z"; return PCE_EINVAL;
    }
}
