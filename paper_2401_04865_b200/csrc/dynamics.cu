// dynamics.cu -- the step on the far side of the hot path: one Brownian-dynamics step of the overdamped
// Langevin equation (eqs. 40-44) with the potential-free hard-sphere interaction written as the pair
// potential of eq. 46, free-draining rigid-body motion of the conductors (eq. 62), and the
// double-layer observables Q'(r), g(r) (eqs. 48-49).  Everything stays on the device: the forces come from
// pce_forces, the new positions go straight into the context (cell lists, hit lists, near field) for the next solve.
// Noise: Philox-4x32-10 (Salmon et al., SC'11), counter = (ion index, step, 0, 0), key = seed -- a counter-based generator, so
// the stream is a pure function of (seed, step, ion) and any other implementation of the same generator reproduces it.
#include "pce_internal.h"

#include <cmath>

namespace {

constexpr int BT = 256;

// ---------------------------------------------------------------- Philox-4x32-10
__device__ __forceinline__ void philox_round(unsigned& c0, unsigned& c1, unsigned& c2, unsigned& c3, unsigned k0, unsigned k1)
{
    const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
}

__device__ __forceinline__ uint4 philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(c0, c1, c2, c3, k0, k1);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;  // Weyl sequence of the key
    }
    return make_uint4(c0, c1, c2, c3);
}

// three standard normal deviates of ion i at time step `step`: Box-Muller on u = (r + 1/2) 2^-32
__device__ __forceinline__ void normals3(unsigned long long seed, unsigned step, unsigned i, double& n0, double& n1, double& n2)
{
    const uint4 r = philox4x32_10(i, step, 0u, 0u, (unsigned)(seed & 0xffffffffull), (unsigned)(seed >> 32));
    const double s = 1.0 / 4294967296.0;
    const double u0 = ((double)r.x + 0.5) * s, u1 = ((double)r.y + 0.5) * s, u2 = ((double)r.z + 0.5) * s, u3 = ((double)r.w + 0.5) * s;
    const double r0 = sqrt(-2.0 * log(u0)), r2 = sqrt(-2.0 * log(u2));
    const double two_pi = 2.0 * PCE_PI;
    n0 = r0 * cos(two_pi * u1);
    n1 = r0 * sin(two_pi * u1);
    n2 = r2 * cos(two_pi * u3);
}

// ---------------------------------------------------------------- hard spheres, eq. 46
struct HsGeom {
    int nc[3], range[3];
    double L[3];
};

// body of caller-order particle p: conductor body of a bead, or a one-particle body per ion
__device__ __forceinline__ int body_id(int p, int nbead, int nbody, const int* __restrict__ body_of)
{
    return p < nbead ? body_of[p] : nbody + (p - nbead);
}

// one thread per particle (sorted order of the 2a-cell binning): f_hs = sum over particles of other bodies with r < 2a of
// gamma (2a - r) / (2 dt) * (x_i - x_j) / r.  Fixed cell and in-cell order: deterministic.
__global__ void __launch_bounds__(BT)
k_hs_forces(int n, HsGeom g, const int* __restrict__ cell_start, const int* __restrict__ cell_of, const int* __restrict__ perm,
            const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs, int nbead, int nbody,
            const int* __restrict__ body_of, double two_a, double pref /* gamma / (2 dt) */, double* __restrict__ fx,
            double* __restrict__ fy, double* __restrict__ fz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int pi = perm[i];
    const int bi = body_id(pi, nbead, nbody, body_of);
    const double xi = xs[i], yi = ys[i], zi = zs[i];
    int cidx = cell_of[pi];
    const int cx = cidx % g.nc[0]; cidx /= g.nc[0];
    const int cy = cidx % g.nc[1], cz = cidx / g.nc[1];
    double ax = 0.0, ay = 0.0, az = 0.0;
    const double r2max = two_a * two_a;
    for (int oz = -g.range[2]; oz <= g.range[2]; ++oz) {
        int kz = cz + oz; double sz = 0.0;
        if (g.nc[2] == 1) { kz = 0; sz = oz * g.L[2]; } else if (kz < 0) { kz += g.nc[2]; sz = -g.L[2]; } else if (kz >= g.nc[2]) { kz -= g.nc[2]; sz = g.L[2]; }
        for (int oy = -g.range[1]; oy <= g.range[1]; ++oy) {
            int ky = cy + oy; double sy = 0.0;
            if (g.nc[1] == 1) { ky = 0; sy = oy * g.L[1]; } else if (ky < 0) { ky += g.nc[1]; sy = -g.L[1]; } else if (ky >= g.nc[1]) { ky -= g.nc[1]; sy = g.L[1]; }
            for (int ox = -g.range[0]; ox <= g.range[0]; ++ox) {
                int kx = cx + ox; double sx = 0.0;
                if (g.nc[0] == 1) { kx = 0; sx = ox * g.L[0]; } else if (kx < 0) { kx += g.nc[0]; sx = -g.L[0]; } else if (kx >= g.nc[0]) { kx -= g.nc[0]; sx = g.L[0]; }
                const int cj = (kz * g.nc[1] + ky) * g.nc[0] + kx;
                const int j1 = cell_start[cj + 1];
                for (int j = cell_start[cj]; j < j1; ++j) {
                    const double dx = xi - (xs[j] + sx), dy = yi - (ys[j] + sy), dz = zi - (zs[j] + sz);
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    if (r2 < r2max && r2 > 0.0) {
                        if (body_id(perm[j], nbead, nbody, body_of) == bi) continue;
                        const double r = sqrt(r2);
                        if (r < two_a) {
                            const double s = pref * (two_a - r) / r;
                            ax += s * dx; ay += s * dy; az += s * dz;
                        }
                    }
                }
            }
        }
    }
    fx[pi] = ax; fy[pi] = ay; fz[pi] = az;
}

__device__ __forceinline__ double wrap1(double x, double L)
{
    x -= L * floor(x / L);
    return x >= L ? 0.0 : x;
}

// ---------------------------------------------------------------- ions: Euler-Maruyama, eqs. 41-44
__global__ void __launch_bounds__(BT)
k_bd_ions(int nion, int nbead, int n, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
          const double* __restrict__ fx, const double* __restrict__ fy, const double* __restrict__ fz, const double* __restrict__ hs,
          const double* __restrict__ noise, pce_bd_params bp, double Lx, double Ly, double Lz, double* __restrict__ xo)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nion) return;
    const int p = nbead + i;
    double n0, n1, n2;
    if (noise) { n0 = noise[i]; n1 = noise[nion + i]; n2 = noise[2 * nion + i]; }
    else normals3(bp.seed, bp.step, (unsigned)i, n0, n1, n2);
    const double mob = bp.dt / bp.gamma, amp = sqrt(2.0 * bp.kT * bp.dt / bp.gamma);
    xo[p] = wrap1(x[p] + (fx[p] + hs[p]) * mob + amp * n0, Lx);
    xo[n + p] = wrap1(y[p] + (fy[p] + hs[n + p]) * mob + amp * n1, Ly);
    xo[2 * n + p] = wrap1(z[p] + (fz[p] + hs[2 * n + p]) * mob + amp * n2, Lz);
}

__device__ __forceinline__ double block_sum(double v, double* sh)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    for (int i = 0; i < BT / 32; ++i) s += sh[i];
    return s;
}

// ---------------------------------------------------------------- bodies: free-draining rigid motion, eq. 62 (one CTA per body)
__global__ void __launch_bounds__(BT)
k_bd_bodies(int n, const int* __restrict__ off, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
            const double* __restrict__ rx, const double* __restrict__ ry, const double* __restrict__ rz, const double* __restrict__ X,
            const double* __restrict__ Y, const double* __restrict__ Z, const double* __restrict__ fx, const double* __restrict__ fy,
            const double* __restrict__ fz, const double* __restrict__ hs, pce_bd_params bp, double Lx, double Ly, double Lz,
            double* __restrict__ xo)
{
    __shared__ double sh[BT / 32];
    __shared__ double R[9], U[3];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    if (!bp.move_bodies) {  // held fixed (reading A13)
        for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) { xo[j] = x[j]; xo[n + j] = y[j]; xo[2 * n + j] = z[j]; }
        return;
    }
    // F, L (eq. 18) of the total force and the rotational resistance gamma sum (r^2 I - r r^T)
    double a[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double f0 = fx[j] + hs[j], f1 = fy[j] + hs[n + j], f2 = fz[j] + hs[2 * n + j], r0 = rx[j], r1 = ry[j], r2 = rz[j];
        a[0] += f0; a[1] += f1; a[2] += f2;
        a[3] += r1 * f2 - r2 * f1; a[4] += r2 * f0 - r0 * f2; a[5] += r0 * f1 - r1 * f0;
        a[6] += r1 * r1 + r2 * r2; a[7] += r0 * r0 + r2 * r2; a[8] += r0 * r0 + r1 * r1;   // I_xx, I_yy, I_zz
        a[9] -= r0 * r1; a[10] -= r0 * r2; a[11] -= r1 * r2;                                  // I_xy, I_xz, I_yz
    }
#pragma unroll
    for (int k = 0; k < 12; ++k) a[k] = block_sum(a[k], sh);
    if (threadIdx.x == 0) {
        const int nb = j1 - j0;
        const double g = bp.gamma;
        U[0] = a[0] / (nb * g) * bp.dt; U[1] = a[1] / (nb * g) * bp.dt; U[2] = a[2] / (nb * g) * bp.dt;
        const double ixx = g * a[6], iyy = g * a[7], izz = g * a[8], ixy = g * a[9], ixz = g * a[10], iyz = g * a[11];
        // cofactors of the symmetric 3 x 3 resistance
        const double c00 = iyy * izz - iyz * iyz, c01 = ixz * iyz - ixy * izz, c02 = ixy * iyz - ixz * iyy;
        const double c11 = ixx * izz - ixz * ixz, c12 = ixy * ixz - ixx * iyz, c22 = ixx * iyy - ixy * ixy;
        const double det = ixx * c00 + ixy * c01 + ixz * c02;
        const double tr3 = (ixx + iyy + izz) / 3.0;
        double w0 = 0.0, w1 = 0.0, w2 = 0.0;  // Omega dt
        if (nb > 1 && det > 1e-10 * tr3 * tr3 * tr3) {  // a single bead or collinear beads: no rotation
            const double s = bp.dt / det;
            w0 = s * (c00 * a[3] + c01 * a[4] + c02 * a[5]);
            w1 = s * (c01 * a[3] + c11 * a[4] + c12 * a[5]);
            w2 = s * (c02 * a[3] + c12 * a[4] + c22 * a[5]);
        }
        // exp([w]_x) = I + A K + B K^2 (Rodrigues), A = sin t / t, B = (1 - cos t) / t^2
        const double t2 = w0 * w0 + w1 * w1 + w2 * w2, t = sqrt(t2);
        double A = 1.0, B = 0.5;
        if (t >= 1e-8) { A = sin(t) / t; const double sh2 = sin(0.5 * t); B = 2.0 * sh2 * sh2 / t2; }
        R[0] = 1.0 - B * (w1 * w1 + w2 * w2); R[1] = -A * w2 + B * w0 * w1;       R[2] = A * w1 + B * w0 * w2;
        R[3] = A * w2 + B * w0 * w1;          R[4] = 1.0 - B * (w0 * w0 + w2 * w2); R[5] = -A * w0 + B * w1 * w2;
        R[6] = -A * w1 + B * w0 * w2;         R[7] = A * w0 + B * w1 * w2;        R[8] = 1.0 - B * (w0 * w0 + w1 * w1);
    }
    __syncthreads();
    const double Xc = X[b] + U[0], Yc = Y[b] + U[1], Zc = Z[b] + U[2];
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double r0 = rx[j], r1 = ry[j], r2 = rz[j];
        xo[j] = wrap1(Xc + (R[0] * r0 + R[1] * r1 + R[2] * r2), Lx);
        xo[n + j] = wrap1(Yc + (R[3] * r0 + R[4] * r1 + R[5] * r2), Ly);
        xo[2 * n + j] = wrap1(Zc + (R[6] * r0 + R[7] * r1 + R[8] * r2), Lz);
    }
}

// ---------------------------------------------------------------- observables, eqs. 48-49
// shell edges exactly as r_lo + k dr (separate multiply and add: no contraction, so that an ion on an edge falls on the same
// side in every implementation of this definition)
__device__ __forceinline__ double shell_edge(double r_lo, double dr, int k) { return __dadd_rn(r_lo, __dmul_rn((double)k, dr)); }

__global__ void __launch_bounds__(BT)
k_profile_bin(int nion, int nbead, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
              const double* __restrict__ q, const double* __restrict__ X, const double* __restrict__ Y, const double* __restrict__ Z,
              int body, double Lx, double Ly, double Lz, double a, double r_lo, double dr, int n_bins, unsigned* __restrict__ cnt,
              double* __restrict__ rho)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nion) return;
    const int p = nbead + i;
    double dx = x[p] - X[body], dy = y[p] - Y[body], dz = z[p] - Z[body];
    dx -= Lx * rint(dx / Lx); dy -= Ly * rint(dy / Ly); dz -= Lz * rint(dz / Lz);
    const double r = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
    const double qi = q[p];
    const int kc = (int)floor((r - r_lo) / dr);
    for (int k = kc - 1; k <= kc + 1; ++k) {  // the shell that holds r, decided by the edge comparisons themselves
        if (k < 0 || k >= n_bins) continue;
        if (r >= shell_edge(r_lo, dr, k) && r < shell_edge(r_lo, dr, k + 1)) {
            if (qi > 0.0) atomicAdd(&cnt[k], 1u);
            else if (qi < 0.0) atomicAdd(&cnt[n_bins + k], 1u);
        }
    }
    if (!rho || qi == 0.0) return;
    const int span = (int)ceil(a / dr) + 2;   // window |r - mid_k| < a
    for (int k = kc - span; k <= kc + span; ++k) {
        if (k < 0 || k >= n_bins) continue;
        const double mid = __dmul_rn(0.5, __dadd_rn(shell_edge(r_lo, dr, k), shell_edge(r_lo, dr, k + 1)));
        if (fabs(r - mid) < a) atomicAdd(&rho[k], qi);
    }
}

// one block: densities, g(r) and the running integral of eq. 48
__global__ void __launch_bounds__(BT)
k_profile_final(int n_bins, int nion, int nbead, const double* __restrict__ q, const int* __restrict__ off, int body, double a, double r_lo,
                double dr, double V, const unsigned* __restrict__ cnt, double* __restrict__ counts, double* __restrict__ g,
                double* __restrict__ rho, double* __restrict__ Qcum)
{
    __shared__ double sh[BT / 32];
    __shared__ double tot[3];
    double np = 0.0, nm = 0.0, Q = 0.0;
    for (int i = threadIdx.x; i < nion; i += blockDim.x) { const double v = q[nbead + i]; np += (v > 0.0); nm += (v < 0.0); }
    for (int j = off[body] + threadIdx.x; j < off[body + 1]; j += blockDim.x) Q += q[j];
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

}  // namespace

void dynamics_free(pce_ctx* c)
{
    bins_free(c->hs);
    cudaFree(c->bd_f); cudaFree(c->bd_x); cudaFree(c->prof_cnt);
    c->bd_f = c->bd_x = nullptr; c->prof_cnt = nullptr; c->prof_cnt_n = 0;
    c->hs_ready = false;
}

// linked cells of edge >= 2a, at most ~2 cells per particle; a dimension with fewer than 3 such cells collapses
// to one cell with explicit periodic images (as for the real-space sum, reading A10)
static int dynamics_alloc(pce_ctx* c)
{
    if (c->hs_ready) return PCE_OK;
    const double two_a = 2.0 * c->p.a;
    const double edge = std::fmax(two_a, std::cbrt(c->V / (2.0 * c->N)));
    int nc[3], range[3];
    for (int d = 0; d < 3; ++d) {
        int n = (int)std::floor(c->p.L[d] / edge);
        if (n > 1024) n = 1024;
        if (n >= 3) { nc[d] = n; range[d] = 1; }
        else { nc[d] = 1; range[d] = (int)std::ceil(two_a / c->p.L[d]); }
    }
    int rc = bins_alloc(c, c->hs, c->N, nc, range);
    if (rc) return rc;
    PCE_CUDA(c, cudaMalloc(&c->bd_f, (size_t)3 * c->N * sizeof(double)));
    PCE_CUDA(c, cudaMalloc(&c->bd_x, (size_t)3 * c->N * sizeof(double)));
    c->bytes += (long long)6 * c->N * 8;
    c->hs_ready = true;
    return PCE_OK;
}

extern "C" int pce_bd_step(pce_ctx* c, const pce_bd_params* bp, const double* fx, const double* fy, const double* fz, const double* noise,
                           double* x, double* y, double* z)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_bd_step before pce_set_system"; return PCE_ESTATE; }
    if (!bp || !fx || !fy || !fz) { c->err = "NULL argument"; return PCE_EINVAL; }
    if (!(bp->dt > 0.0) || !(bp->gamma > 0.0) || !(bp->kT >= 0.0)) { c->err = "pce_bd_step: need dt > 0, gamma > 0, kT >= 0"; return PCE_EINVAL; }
    int rc = dynamics_alloc(c);
    if (rc) return rc;
    TimingScope timed(c);  // the step's passes (hard spheres under "other", the rebuild under cells / real) in pce_get_timings
    const int N = c->N;
    {
        PassTimer t(c, PASS_OTHER);
        if ((rc = bins_build(c, c->hs, c->x, c->y, c->z))) return rc;
        HsGeom g;
        for (int d = 0; d < 3; ++d) { g.nc[d] = c->hs.nc[d]; g.range[d] = c->hs.range[d]; g.L[d] = c->p.L[d]; }
        k_hs_forces<<<cdiv(N, BT), BT, 0, c->st>>>(N, g, c->hs.cell_start, c->hs.cell_of, c->hs.perm, c->hs.xs, c->hs.ys, c->hs.zs, c->Nbead,
                                                  c->Nbody, c->body_of, 2.0 * c->p.a, bp->gamma / (2.0 * bp->dt), c->bd_f, c->bd_f + N,
                                                  c->bd_f + 2 * (size_t)N);
        c->launches++;
        if (c->Nion > 0) {
            k_bd_ions<<<cdiv(c->Nion, BT), BT, 0, c->st>>>(c->Nion, c->Nbead, N, c->x, c->y, c->z, fx, fy, fz, c->bd_f, noise, *bp, c->p.L[0],
                                                          c->p.L[1], c->p.L[2], c->bd_x);
            c->launches++;
        }
        if (c->Nbody > 0) {
            k_bd_bodies<<<c->Nbody, BT, 0, c->st>>>(N, c->body_off, c->x, c->y, c->z, c->rx, c->ry, c->rz, c->X, c->Y, c->Z, fx, fy, fz, c->bd_f,
                                                   *bp, c->p.L[0], c->p.L[1], c->p.L[2], c->bd_x);
            c->launches++;
        }
        PCE_CUDA(c, cudaGetLastError());
    }
    if ((rc = positions_update(c, c->bd_x, c->bd_x + N, c->bd_x + 2 * (size_t)N))) return rc;
    if (x) PCE_CUDA(c, cudaMemcpyAsync(x, c->x, (size_t)N * 8, cudaMemcpyDeviceToDevice, c->st));
    if (y) PCE_CUDA(c, cudaMemcpyAsync(y, c->y, (size_t)N * 8, cudaMemcpyDeviceToDevice, c->st));
    if (z) PCE_CUDA(c, cudaMemcpyAsync(z, c->z, (size_t)N * 8, cudaMemcpyDeviceToDevice, c->st));
    return PCE_OK;
}

extern "C" int pce_radial_profile(pce_ctx* c, int body, const double* q, double r_lo, int n_bins, double* counts, double* g, double* rho,
                                  double* Qcum)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_radial_profile before pce_set_system"; return PCE_ESTATE; }
    if (!q || body < 0 || body >= c->Nbody || n_bins <= 0 || !(r_lo >= 0.0)) { c->err = "pce_radial_profile: bad arguments"; return PCE_EINVAL; }
    if (Qcum && !rho) { c->err = "pce_radial_profile: Qcum needs rho"; return PCE_EINVAL; }
    TimingScope timed(c);
    PassTimer t(c, PASS_OTHER);
    if (c->prof_cnt_n < 2 * n_bins) {
        cudaFree(c->prof_cnt);
        c->prof_cnt = nullptr; c->prof_cnt_n = 0;
        PCE_CUDA(c, cudaMalloc(&c->prof_cnt, (size_t)2 * n_bins * sizeof(unsigned)));
        c->prof_cnt_n = 2 * n_bins;
    }
    PCE_CUDA(c, cudaMemsetAsync(c->prof_cnt, 0, (size_t)2 * n_bins * sizeof(unsigned), c->st));
    if (rho) PCE_CUDA(c, cudaMemsetAsync(rho, 0, (size_t)n_bins * sizeof(double), c->st));
    const double dr = 0.1 * c->p.a;
    if (c->Nion > 0) {
        k_profile_bin<<<cdiv(c->Nion, BT), BT, 0, c->st>>>(c->Nion, c->Nbead, c->x, c->y, c->z, q, c->X, c->Y, c->Z, body, c->p.L[0], c->p.L[1],
                                                          c->p.L[2], c->p.a, r_lo, dr, n_bins, c->prof_cnt, rho);
        c->launches++;
    }
    k_profile_final<<<1, BT, 0, c->st>>>(n_bins, c->Nion, c->Nbead, q, c->body_off, body, c->p.a, r_lo, dr, c->V, c->prof_cnt, counts, g, rho, Qcum);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
