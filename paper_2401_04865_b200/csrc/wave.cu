// wave.cu -- wave-space part of the Ewald split by the spectral Ewald method
// (PAPER.md:202-268), steps 3-5: FFT (cuFFT, the only library call), scaling by
// j0(ka)^2 exp(-(1-eta)k^2/4xi^2)/k^2 (eq. 26), inverse FFT.  Spreading (eq. 25)
// and gather (eq. 27) are in wave_bricks.cu.
//
// Window (reading G4): w(r) = prod_d (2/(P h_d^2))^(1/2) exp(-2 pi u_d^2 / P),
// u = r/h, i.e. eq. 25 with eta_d = h_d^2 xi^2 P/pi (eq. 31).  Spread and gather use the
// same UNNORMALISED weights W = exp(-aw u^2); every constant (window norm^2, h^3 of the
// quadrature, 1/V, 1/eps_f, cuFFT's missing 1/N) is folded into the scaling pass.
#include "pce_internal.h"

// ---------------------------------------------------------------- scale (eq. 26)
// The Green's function depends on (|kx|, |ky|, |kz|) only, so one thread evaluates it once (sqrt, sin, exp,
// two divisions: ~150 fp64 instructions) and applies it to the up to four mirror points (+-ky, +-kz) of the
// half spectrum: the pass is then bound by its 32 bytes per complex mesh point of HBM traffic, not by the fp64 pipe.
__global__ void __launch_bounds__(256)
k_scale(WaveConst wc, cufftDoubleComplex* __restrict__ gk, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    const int nxh = wc.Nxh, ny = wc.Ng[1], nz = wc.Ng[2];
    const int hy = ny / 2 + 1, hz = nz / 2 + 1;  // iy in [0, ny/2], iz in [0, nz/2]; mirrors ny - iy, nz - iz
    const size_t total = (size_t)nxh * hy * hz;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(idx % nxh);
        const size_t rest = idx / nxh;
        const int iy = (int)(rest % hy), iz = (int)(rest / hy);
        const double kx = wc.kfac[0] * ix, ky = wc.kfac[1] * iy, kz = wc.kfac[2] * iz;  // fftfreq ordering (reading A6)
        const double kx2 = kx * kx, ky2 = ky * ky, kz2 = kz * kz;
        const double k2 = kx2 + ky2 + kz2;
        double f = 0.0;  // k = 0 removed
        if (k2 > 0.0) {
            const double ka = sqrt(k2) * wc.a;
            const double j0 = (ka < 1e-4) ? 1.0 - ka * ka * (1.0 / 6.0) : sin(ka) / ka;
            f = wc.scale_norm * j0 * j0 * exp(-(wc.gexp[0] * kx2 + wc.gexp[1] * ky2 + wc.gexp[2] * kz2)) / k2;
        }
        const int my = (iy == 0 || 2 * iy == ny) ? -1 : ny - iy;  // mirror rows (none for the self-mirrored planes)
        const int mz = (iz == 0 || 2 * iz == nz) ? -1 : nz - iz;
        cufftDoubleComplex* p00 = gk + ((size_t)iz * ny + iy) * nxh + ix;
        cufftDoubleComplex* p10 = (my >= 0) ? gk + ((size_t)iz * ny + my) * nxh + ix : nullptr;
        cufftDoubleComplex* p01 = (mz >= 0) ? gk + ((size_t)mz * ny + iy) * nxh + ix : nullptr;
        cufftDoubleComplex* p11 = (my >= 0 && mz >= 0) ? gk + ((size_t)mz * ny + my) * nxh + ix : nullptr;
        cufftDoubleComplex v00 = *p00, v10 = {0, 0}, v01 = {0, 0}, v11 = {0, 0};
        if (p10) v10 = *p10;
        if (p01) v01 = *p01;
        if (p11) v11 = *p11;
        v00.x *= f; v00.y *= f;
        *p00 = v00;
        if (p10) { v10.x *= f; v10.y *= f; *p10 = v10; }
        if (p01) { v01.x *= f; v01.y *= f; *p01 = v01; }
        if (p11) { v11.x *= f; v11.y *= f; *p11 = v11; }
    }
}

int wave_fft_scale_ifft(pce_ctx* c)
{
    {
        PassTimer t(c, PASS_FFT);
        if (cufftExecD2Z(c->planF, c->grid, c->gridk) != CUFFT_SUCCESS) { c->err = "cufftExecD2Z failed"; return PCE_ECUFFT; }
    }
    if (c->use_zfft) {
        PassTimer t(c, PASS_SCALE);  // z FFT + Green's function + inverse z FFT in one pass over the half spectrum
        int rc = zfft_scale(c);
        if (rc) return rc;
    } else {
        PassTimer t(c, PASS_SCALE);
        const size_t total = (size_t)c->wk.Nxh * (c->wk.Ng[1] / 2 + 1) * (c->wk.Ng[2] / 2 + 1);
        const int blocks = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
        k_scale<<<blocks, 256, 0, c->st>>>(c->wk, c->gridk, c->skip_flag);
        c->launches++;
        PCE_CUDA(c, cudaGetLastError());
    }
    {
        PassTimer t(c, PASS_IFFT);
        if (cufftExecZ2D(c->planB, c->gridk, c->grid) != CUFFT_SUCCESS) { c->err = "cufftExecZ2D failed"; return PCE_ECUFFT; }
    }
    return PCE_OK;
}
