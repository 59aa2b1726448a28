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
k_scale(WaveConst wc, const cufftDoubleComplex* gin, cufftDoubleComplex* gout, int deriv, const int* __restrict__ skip)
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
        // ik differentiation (deriv = 0, 1, 2): times -i k_d, k_d signed (the mirror rows carry -k_y, -k_z), 0 at the Nyquist mode
        double kd = 0.0;
        if (deriv == 0) kd = (2 * ix == wc.Ng[0]) ? 0.0 : kx;
        if (deriv == 1) kd = (2 * iy == ny) ? 0.0 : ky;
        if (deriv == 2) kd = (2 * iz == nz) ? 0.0 : kz;
        const int my = (iy == 0 || 2 * iy == ny) ? -1 : ny - iy;  // mirror rows (none for the self-mirrored planes)
        const int mz = (iz == 0 || 2 * iz == nz) ? -1 : nz - iz;
        const size_t o00 = ((size_t)iz * ny + iy) * nxh + ix;
        const size_t o10 = (my >= 0) ? ((size_t)iz * ny + my) * nxh + ix : o00;
        const size_t o01 = (mz >= 0) ? ((size_t)mz * ny + iy) * nxh + ix : o00;
        const size_t o11 = (my >= 0 && mz >= 0) ? ((size_t)mz * ny + my) * nxh + ix : o00;
        cufftDoubleComplex v00 = gin[o00], v10 = {0, 0}, v01 = {0, 0}, v11 = {0, 0};
        if (my >= 0) v10 = gin[o10];
        if (mz >= 0) v01 = gin[o01];
        if (my >= 0 && mz >= 0) v11 = gin[o11];
        auto apply = [&](cufftDoubleComplex v, double sgn) {
            cufftDoubleComplex r;
            if (deriv < 0) { r.x = v.x * f; r.y = v.y * f; }
            else { const double g = f * kd * sgn; r.x = v.y * g; r.y = -v.x * g; }  // -i k (x + i y) = k (y - i x)
            return r;
        };
        const double sy = (deriv == 1) ? -1.0 : 1.0, sz = (deriv == 2) ? -1.0 : 1.0;
        gout[o00] = apply(v00, 1.0);
        if (my >= 0) gout[o10] = apply(v10, sy);
        if (mz >= 0) gout[o01] = apply(v01, sz);
        if (my >= 0 && mz >= 0) gout[o11] = apply(v11, sy * sz);
    }
}

int wave_forward(pce_ctx* c)
{
    PassTimer t(c, PASS_FFT);
    if (c->use_fftxy) return fftxy_forward(c, c->gridk);
    if (cufftExecD2Z(c->planF, c->grid, c->gridk) != CUFFT_SUCCESS) { c->err = "cufftExecD2Z failed"; return PCE_ECUFFT; }
    return PCE_OK;
}

// deriv < 0: in place on gridk; deriv >= 0: gridk -> gridk2 (the forward spectrum survives for the next component)
int wave_scale_inverse(pce_ctx* c, int deriv)
{
    cufftDoubleComplex* out = c->gridk;
    if (deriv >= 0) {
        if (!c->gridk2) {
            const size_t nk = (size_t)c->wk.Nxh * c->wk.Ng[1] * c->wk.Ng[2];
            if (cudaMalloc(&c->gridk2, nk * sizeof(cufftDoubleComplex)) != cudaSuccess) { c->err = "out of device memory for the second spectrum (ik fields)"; return PCE_ENOMEM; }
            c->bytes += (long long)(nk * 16); c->bytes_base += (long long)(nk * 16);
        }
        out = c->gridk2;
    }
    if (c->use_zfft) {
        PassTimer t(c, PASS_SCALE);  // z FFT + Green's function + inverse z FFT in one pass over the half spectrum
        int rc = zfft_scale(c, c->gridk, out, deriv);
        if (rc) return rc;
    } else {
        PassTimer t(c, PASS_SCALE);
        const size_t total = (size_t)c->wk.Nxh * (c->wk.Ng[1] / 2 + 1) * (c->wk.Ng[2] / 2 + 1);
        const int blocks = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
        k_scale<<<blocks, 256, 0, c->st>>>(c->wk, c->gridk, out, deriv, c->skip_flag);
        c->launches++;
        PCE_CUDA(c, cudaGetLastError());
    }
    {
        PassTimer t(c, PASS_IFFT);
        if (c->use_fftxy) return fftxy_inverse(c, out);
        if (cufftExecZ2D(c->planB, out, c->grid) != CUFFT_SUCCESS) { c->err = "cufftExecZ2D failed"; return PCE_ECUFFT; }
    }
    return PCE_OK;
}

int wave_fft_scale_ifft(pce_ctx* c)
{
    int rc = wave_forward(c);
    if (!rc) rc = wave_scale_inverse(c, -1);
    return rc;
}
