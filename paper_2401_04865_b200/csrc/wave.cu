// wave.cu -- wave-space part of the Ewald split by the spectral Ewald method
// (PAPER.md:202-268): Gaussian spreading H(x) (eq. 25), FFT (cuFFT, the only
// library call), scaling by j0(ka)^2 exp(-(1-eta)k^2/4xi^2)/k^2 (eq. 26),
// inverse FFT, Gaussian gather by the trapezoid rule (eq. 27).
//
// Window (reading G4): w(r) = prod_d (2/(P h_d^2))^(1/2) exp(-2 pi u_d^2 / P),
// u = r/h, i.e. eq. 25 with eta_d = h_d^2 xi^2 P/pi (eq. 31).  Spread and gather use the
// same UNNORMALISED weights W = exp(-aw u^2); every constant (window norm^2, h^3 of the
// quadrature, 1/V, 1/eps_f, cuFFT's missing 1/N) is folded into the scaling pass.
#include "pce_internal.h"

constexpr int SG_WARPS = 4;

// weights, wrapped grid indices and offsets of one particle, per warp, in shared memory
struct WarpWin {
    double w[3][32];
    double u[3][32];
    int g[3][32];
};

__device__ __forceinline__ void window_setup(const WaveConst& wc, WarpWin& win, int lane, double x, double y, double z)
{
    const int P = wc.P;
    for (int t = lane; t < 3 * P; t += 32) {
        const int d = t / P, j = t - d * P;
        const double xd = (d == 0 ? x : (d == 1 ? y : z)) * wc.inv_h[d];
        const int i0 = (int)floor(xd);
        int g = i0 - P / 2 + 1 + j;  // even P: floor(x/h) - P/2 + 1 ... floor(x/h) + P/2 (reading A5)
        const double u = (double)g - xd;
        const int ng = wc.Ng[d];
        if (g < 0) g += ng;
        if (g >= ng) g -= ng;
        win.w[d][j] = exp(-wc.aw * u * u);
        win.u[d][j] = u;
        win.g[d][j] = g;
    }
    __syncwarp();
}

// ---------------------------------------------------------------- spread (eq. 25)
__global__ void __launch_bounds__(SG_WARPS * 32)
k_spread_atomic(int n, WaveConst wc, const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                const double* __restrict__ qs, double* __restrict__ grid)
{
    __shared__ WarpWin wins[SG_WARPS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * SG_WARPS + warp;
    if (i >= n) return;
    const double q = qs[i];
    if (q == 0.0) return;
    WarpWin& win = wins[warp];
    window_setup(wc, win, lane, xs[i], ys[i], zs[i]);
    const int P = wc.P, PP = P * P;
    const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
    for (int jz = 0; jz < P; ++jz) {
        const double qz = q * win.w[2][jz];
        const size_t oz = (size_t)win.g[2][jz] * Ny;
        for (int t = lane; t < PP; t += 32) {
            const int jy = t / P, jx = t - jy * P;
            atomicAdd(&grid[(oz + win.g[1][jy]) * Nx + win.g[0][jx]], qz * win.w[1][jy] * win.w[0][jx]);
        }
    }
}

int wave_spread(pce_ctx* c, const Bins& b)
{
    PassTimer t(c, PASS_SPREAD);
    const size_t ng = (size_t)c->wk.Ng[0] * c->wk.Ng[1] * c->wk.Ng[2];
    PCE_CUDA(c, cudaMemsetAsync(c->grid, 0, ng * sizeof(double), c->st));
    if (b.n == 0) return PCE_OK;
    k_spread_atomic<<<cdiv(b.n, SG_WARPS), SG_WARPS * 32, 0, c->st>>>(b.n, c->wk, b.xs, b.ys, b.zs, b.qs, c->grid);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// ---------------------------------------------------------------- scale (eq. 26)
__global__ void __launch_bounds__(256)
k_scale(WaveConst wc, cufftDoubleComplex* __restrict__ gk)
{
    const size_t nxh = wc.Nxh, ny = wc.Ng[1], nz = wc.Ng[2];
    const size_t total = nxh * ny * nz;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(idx % nxh);
        const size_t rest = idx / nxh;
        const int iy = (int)(rest % ny), iz = (int)(rest / ny);
        const int fy = (iy <= (int)ny / 2) ? iy : iy - (int)ny;  // fftfreq ordering (reading A6)
        const int fz = (iz <= (int)nz / 2) ? iz : iz - (int)nz;
        const double kx = wc.kfac[0] * ix, ky = wc.kfac[1] * fy, kz = wc.kfac[2] * fz;
        const double kx2 = kx * kx, ky2 = ky * ky, kz2 = kz * kz;
        const double k2 = kx2 + ky2 + kz2;
        double f = 0.0;  // k = 0 removed
        if (k2 > 0.0) {
            const double ka = sqrt(k2) * wc.a;
            const double j0 = (ka < 1e-4) ? 1.0 - ka * ka * (1.0 / 6.0) : sin(ka) / ka;
            f = wc.scale_norm * j0 * j0 * exp(-(wc.gexp[0] * kx2 + wc.gexp[1] * ky2 + wc.gexp[2] * kz2)) / k2;
        }
        cufftDoubleComplex v = gk[idx];
        v.x *= f; v.y *= f;
        gk[idx] = v;
    }
}

int wave_fft_scale_ifft(pce_ctx* c)
{
    {
        PassTimer t(c, PASS_FFT);
        if (cufftExecD2Z(c->planF, c->grid, c->gridk) != CUFFT_SUCCESS) { c->err = "cufftExecD2Z failed"; return PCE_ECUFFT; }
    }
    {
        PassTimer t(c, PASS_SCALE);
        const size_t total = (size_t)c->wk.Nxh * c->wk.Ng[1] * c->wk.Ng[2];
        const int blocks = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
        k_scale<<<blocks, 256, 0, c->st>>>(c->wk, c->gridk);
        c->launches++;
        PCE_CUDA(c, cudaGetLastError());
    }
    {
        PassTimer t(c, PASS_IFFT);
        if (cufftExecZ2D(c->planB, c->gridk, c->grid) != CUFFT_SUCCESS) { c->err = "cufftExecZ2D failed"; return PCE_ECUFFT; }
    }
    return PCE_OK;
}

// ---------------------------------------------------------------- gather (eq. 27)
template <bool FIELD>
__global__ void __launch_bounds__(SG_WARPS * 32)
k_gather_warp(int n, WaveConst wc, const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
              const double* __restrict__ grid, double* __restrict__ psi, double* __restrict__ ex, double* __restrict__ ey,
              double* __restrict__ ez)
{
    __shared__ WarpWin wins[SG_WARPS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * SG_WARPS + warp;
    if (i >= n) return;
    WarpWin& win = wins[warp];
    window_setup(wc, win, lane, xs[i], ys[i], zs[i]);
    const int P = wc.P, PP = P * P;
    const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
    double s0 = 0, sx = 0, sy = 0, sz = 0;
    for (int jz = 0; jz < P; ++jz) {
        const double wz = win.w[2][jz];
        const size_t oz = (size_t)win.g[2][jz] * Ny;
        double p0 = 0, px = 0, py = 0;
        for (int t = lane; t < PP; t += 32) {
            const int jy = t / P, jx = t - jy * P;
            const double v = grid[(oz + win.g[1][jy]) * Nx + win.g[0][jx]] * win.w[1][jy] * win.w[0][jx];
            p0 += v;
            if (FIELD) { px += v * win.u[0][jx]; py += v * win.u[1][jy]; }
        }
        s0 += wz * p0;
        if (FIELD) { sx += wz * px; sy += wz * py; sz += wz * win.u[2][jz] * p0; }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, off);
        if (FIELD) {
            sx += __shfl_xor_sync(0xffffffffu, sx, off);
            sy += __shfl_xor_sync(0xffffffffu, sy, off);
            sz += __shfl_xor_sync(0xffffffffu, sz, off);
        }
    }
    if (lane == 0) {
        psi[i] = s0;
        if (FIELD) {  // E = -grad_alpha: dW/dx_alpha = +grad_fac u W
            ex[i] = -wc.grad_fac[0] * sx; ey[i] = -wc.grad_fac[1] * sy; ez[i] = -wc.grad_fac[2] * sz;
        }
    }
}

int wave_gather(pce_ctx* c, const Bins& b, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s)
{
    if (b.n == 0) return PCE_OK;
    PassTimer t(c, PASS_GATHER);
    const int blocks = cdiv(b.n, SG_WARPS);
    if (field)
        k_gather_warp<true><<<blocks, SG_WARPS * 32, 0, c->st>>>(b.n, c->wk, b.xs, b.ys, b.zs, c->grid, psi_s, ex_s, ey_s, ez_s);
    else
        k_gather_warp<false><<<blocks, SG_WARPS * 32, 0, c->st>>>(b.n, c->wk, b.xs, b.ys, b.zs, c->grid, psi_s, nullptr, nullptr, nullptr);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
