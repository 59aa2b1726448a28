// profile_static.cu -- pce_radial_profile_static: the double-layer observables of pce_radial_profile (eqs. 48-49,
// PAPER.md:413-434) for callers that must not allocate device memory.
//
// Who that is.  The paper's own code runs as a plug-in of a molecular-dynamics engine, and an analysis hook of
// that kind is the typical caller of this observable: it runs every few time steps inside a host program whose own pool has
// already claimed the device memory (a cudaMalloc there may simply fail half-way through a run), and it runs between the
// engine's kernels, where cudaMalloc / cudaFree would make the whole device wait.  pce_radial_profile needs a pce_ctx (hundreds
// of megabytes of workspace at the sizes of the paper) and grows a counter buffer with cudaMalloc when n_bins grows.  This entry
// point needs neither: the caller passes the ions, the body's bead charges and the output arrays, and the only scratch memory
// -- the integer shell counters the ions are binned into with atomics -- is the fixed array below, part of the loaded library
// image.  Nothing in this file calls cudaMalloc, cudaFree or a library routine that allocates.
//
// The arithmetic is that of k_profile_bin / k_profile_final in dynamics.cu, restated here with the ions, the centre and the
// bead charges as direct arguments (those kernels read them out of a context), so that both paths put every ion in the same
// shell and agree to the rounding of the fp64 atomics on rho.
#include "pce_internal.h"

#include <cstdio>
#include <mutex>

// The shell counters: cations [0, n_bins), anions [n_bins, 2 n_bins).  2 x 16384 x 4 B = 128 KiB, held by every GPU that loads
// libpce.so until the process exits.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device
// address and must never be handed to a kernel or to cudaMemset; device code may name it directly.
static __device__ __align__(256) unsigned g_shell_counters[2 * PCE_PROFILE_STATIC_MAX_BINS];

namespace {

constexpr int BT = 256;
constexpr int MAX_DEVICES = 64;

std::mutex g_setup_lock;
unsigned* g_counters_of_device[MAX_DEVICES] = {nullptr};  // device address of g_shell_counters, per CUDA device ordinal

__device__ __forceinline__ double shell_edge(double r_lo, double dr, int k) { return __dadd_rn(r_lo, __dmul_rn((double)k, dr)); }

__device__ __forceinline__ double block_sum(double v, double* sh)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < BT / 32; ++w) s += sh[w];
    return s;
}

// one thread per ion: the shell that holds its minimum-image distance from the centre (eq. 49's count) and its share of the
// 2a-wide sliding window of the charge density
__global__ void __launch_bounds__(BT)
k_profile_bin_static(int nion, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                     const double* __restrict__ q, double cx, double cy, double cz, double Lx, double Ly, double Lz, double a,
                     double r_lo, double dr, int n_bins, unsigned* __restrict__ cnt, double* __restrict__ rho)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nion) return;
    double dx = x[i] - cx, dy = y[i] - cy, dz = z[i] - cz;
    dx -= Lx * rint(dx / Lx); dy -= Ly * rint(dy / Ly); dz -= Lz * rint(dz / Lz);
    const double r = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
    const double qi = q[i];
    const int kc = (int)floor((r - r_lo) / dr);
    for (int k = kc - 1; k <= kc + 1; ++k) {  // decided by the edge comparisons themselves, as in dynamics.cu
        if (k < 0 || k >= n_bins) continue;
        if (r >= shell_edge(r_lo, dr, k) && r < shell_edge(r_lo, dr, k + 1)) {
            if (qi > 0.0) atomicAdd(&cnt[k], 1u);
            else if (qi < 0.0) atomicAdd(&cnt[n_bins + k], 1u);
        }
    }
    if (!rho || qi == 0.0) return;
    const int span = (int)ceil(a / dr) + 2;
    for (int k = kc - span; k <= kc + span; ++k) {
        if (k < 0 || k >= n_bins) continue;
        const double mid = __dmul_rn(0.5, __dadd_rn(shell_edge(r_lo, dr, k), shell_edge(r_lo, dr, k + 1)));
        if (fabs(r - mid) < a) atomicAdd(&rho[k], qi);
    }
}

// one block: species totals, the body's net charge, then counts -> g(r) (eq. 49), rho / 2a and the running integral of eq. 48
__global__ void __launch_bounds__(BT)
k_profile_final_static(int n_bins, int nion, const double* __restrict__ q_ion, int nbead, const double* __restrict__ q_bead, double a,
                       double r_lo, double dr, double V, const unsigned* __restrict__ cnt, double* __restrict__ counts,
                       double* __restrict__ g, double* __restrict__ rho, double* __restrict__ Qcum)
{
    __shared__ double sh[BT / 32];
    __shared__ double tot[3];
    double np = 0.0, nm = 0.0, Q = 0.0;
    for (int i = threadIdx.x; i < nion; i += blockDim.x) { const double v = q_ion[i]; np += (v > 0.0); nm += (v < 0.0); }
    for (int j = threadIdx.x; j < nbead; j += blockDim.x) Q += q_bead[j];
    np = block_sum(np, sh); nm = block_sum(nm, sh); Q = block_sum(Q, sh);
    if (threadIdx.x == 0) { tot[0] = np; tot[1] = nm; tot[2] = Q; }
    __syncthreads();
    for (int k = threadIdx.x; k < n_bins; k += blockDim.x) {
        const double lo = shell_edge(r_lo, dr, k), hi = shell_edge(r_lo, dr, k + 1);
        const double shell = 4.0 * PCE_PI / 3.0 * (hi * hi * hi - lo * lo * lo);
        for (int s = 0; s < 2; ++s) {
            const double cv = (double)cnt[s * n_bins + k];
            if (counts) counts[s * n_bins + k] = cv;
            if (g) g[s * n_bins + k] = cv / fmax(tot[s] / V * shell, 1e-300);
        }
        if (rho) rho[k] = rho[k] / (2.0 * a);
    }
    __syncthreads();
    if (threadIdx.x == 0 && Qcum && rho) {
        double run = 0.0;
        for (int k = 0; k < n_bins; ++k) { run += rho[k]; Qcum[k] = tot[2] + run * dr; }
    }
}

int fail(char* err, int err_len, int code, const char* fmt, long long v0 = 0, long long v1 = 0)
{
    if (err && err_len > 0) std::snprintf(err, (size_t)err_len, fmt, v0, v1);
    return code;
}

// Device address of g_shell_counters on the CURRENT device, looked up on the first call made with that device current.
int counters_of_current_device(unsigned** out, char* err, int err_len)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        if (err && err_len > 0) std::snprintf(err, (size_t)err_len, "pce_radial_profile_static: cudaGetDevice: %s", cudaGetErrorString(e));
        return PCE_ECUDA;
    }
    if (dev < 0 || dev >= MAX_DEVICES) return fail(err, err_len, PCE_EINVAL, "pce_radial_profile_static: device ordinal %lld is beyond the %lld this entry point keeps addresses for", dev, MAX_DEVICES);
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_counters_of_device[dev]) {
        unsigned* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_shell_counters);
        if (e != cudaSuccess || !p) {
            if (err && err_len > 0) std::snprintf(err, (size_t)err_len, "pce_radial_profile_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return PCE_ECUDA;
        }
        g_counters_of_device[dev] = p;
    }
    *out = g_counters_of_device[dev];
    return PCE_OK;
}

}  // namespace

extern "C" int pce_radial_profile_static(void* stream, int n_ion, const double* x, const double* y, const double* z, const double* q_ion,
                                         int n_bead, const double* q_bead, const double centre[3], const double L[3], double a,
                                         double r_lo, int n_bins, double* counts, double* g, double* rho, double* Qcum, char* err,
                                         int err_len)
{
    if (err && err_len > 0) err[0] = '\0';
    if (n_bins > PCE_PROFILE_STATIC_MAX_BINS)
        return fail(err, err_len, PCE_EINVAL, "pce_radial_profile_static: n_bins = %lld exceeds PCE_PROFILE_STATIC_MAX_BINS = %lld (the fixed counter array); use fewer shells per call or pce_radial_profile", n_bins, PCE_PROFILE_STATIC_MAX_BINS);
    if (n_bins <= 0 || n_ion < 0 || n_bead < 0) return fail(err, err_len, PCE_EINVAL, "pce_radial_profile_static: need n_bins > 0, n_ion >= 0, n_bead >= 0");
    if (n_ion > 0 && (!x || !y || !z || !q_ion)) return fail(err, err_len, PCE_EINVAL, "pce_radial_profile_static: NULL ion array");
    if (n_bead > 0 && !q_bead) return fail(err, err_len, PCE_EINVAL, "pce_radial_profile_static: NULL q_bead");
    if (!centre || !L || !(L[0] > 0.0) || !(L[1] > 0.0) || !(L[2] > 0.0) || !(a > 0.0) || !(r_lo >= 0.0))
        return fail(err, err_len, PCE_EINVAL, "pce_radial_profile_static: need centre, L > 0, a > 0, r_lo >= 0");
    if (Qcum && !rho) return fail(err, err_len, PCE_EINVAL, "pce_radial_profile_static: Qcum needs rho");

    unsigned* cnt = nullptr;
    int rc = counters_of_current_device(&cnt, err, err_len);
    if (rc) return rc;

    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps what the previous call left in it: the counters of this call's shells start from zero
    cudaError_t e = cudaMemsetAsync(cnt, 0, (size_t)2 * n_bins * sizeof(unsigned), st);
    if (e == cudaSuccess && rho) e = cudaMemsetAsync(rho, 0, (size_t)n_bins * sizeof(double), st);
    if (e == cudaSuccess) {
        const double dr = 0.1 * a;
        if (n_ion > 0)
            k_profile_bin_static<<<cdiv(n_ion, BT), BT, 0, st>>>(n_ion, x, y, z, q_ion, centre[0], centre[1], centre[2], L[0], L[1], L[2], a,
                                                                r_lo, dr, n_bins, cnt, rho);
        k_profile_final_static<<<1, BT, 0, st>>>(n_bins, n_ion, q_ion, n_bead, q_bead, a, r_lo, dr, L[0] * L[1] * L[2], cnt, counts, g, rho,
                                                Qcum);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (err && err_len > 0) std::snprintf(err, (size_t)err_len, "pce_radial_profile_static: %s", cudaGetErrorString(e));
        return PCE_ECUDA;
    }
    return PCE_OK;
}
