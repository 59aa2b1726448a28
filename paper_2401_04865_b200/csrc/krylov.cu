// krylov.cu -- rigid-body bookkeeping (Sigma of eq. 13 / eq. 52 as contiguous
// bead ranges), the on-device conjugate-gradient solve of the induced-charge
// saddle-point system eq. 13 in its per-body-mean-projected SPD
// form, and the moments / forces / torques / energies of eqs. 14, 16-18
// (PAPER.md:137-163).  All reductions have a fixed order (deterministic).
#include "pce_internal.h"

constexpr int BT = 256;  // threads of the per-body / reduction blocks

__device__ __forceinline__ double block_sum(double v, double* sh)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    double s = 0.0;
    const int nw = (blockDim.x + 31) >> 5;
    for (int i = 0; i < nw; ++i) s += sh[i];
    return s;
}

// out[0] = sum(in[0..n))   (single block, fixed order)
__global__ void __launch_bounds__(1024) k_sum(const double* __restrict__ in, long long n, double* __restrict__ out)
{
    __shared__ double sh[32];
    double v = 0.0;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) v += in[i];
    const double s = block_sum(v, sh);
    if (threadIdx.x == 0) out[0] = s;
}

static int sum_to(pce_ctx* c, const double* in, long long n, double* out)
{
    k_sum<<<1, 1024, 0, c->st>>>(in, n, out);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

__device__ __forceinline__ double min_img(double d, double L) { return d - L * floor(d / L + 0.5); }

// ---------------------------------------------------------------- body centres and r_ij (eq. 12)
__global__ void __launch_bounds__(BT)
k_body_centres(const int* __restrict__ off, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
               double Lx, double Ly, double Lz, double* __restrict__ rx, double* __restrict__ ry, double* __restrict__ rz,
               double* __restrict__ X, double* __restrict__ Y, double* __restrict__ Z)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    if (j1 <= j0) { if (threadIdx.x == 0) { X[b] = Y[b] = Z[b] = 0.0; } return; }
    const double x0 = x[j0], y0 = y[j0], z0 = z[j0];
    double sx = 0, sy = 0, sz = 0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        sx += min_img(x[j] - x0, Lx); sy += min_img(y[j] - y0, Ly); sz += min_img(z[j] - z0, Lz);
    }
    const double inv = 1.0 / (j1 - j0);
    const double mx = block_sum(sx, sh) * inv;
    const double my = block_sum(sy, sh) * inv;
    const double mz = block_sum(sz, sh) * inv;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        rx[j] = min_img(x[j] - x0, Lx) - mx; ry[j] = min_img(y[j] - y0, Ly) - my; rz[j] = min_img(z[j] - z0, Lz) - mz;
    }
    if (threadIdx.x == 0) { X[b] = x0 + mx; Y[b] = y0 + my; Z[b] = z0 + mz; }
}

int bodies_setup(pce_ctx* c)
{
    if (c->Nbody == 0) return PCE_OK;
    k_body_centres<<<c->Nbody, BT, 0, c->st>>>(c->body_off, c->x, c->y, c->z, c->p.L[0], c->p.L[1], c->p.L[2], c->rx, c->ry, c->rz,
                                             c->X, c->Y, c->Z);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// ---------------------------------------------------------------- CG pieces
// initial charges: beads Q_i/N_i (or the caller's guess re-centred so that sum_j q_ij = Q_i), ions fixed
__global__ void __launch_bounds__(BT)
k_init_q(const int* __restrict__ off, const double* __restrict__ Qb, int warm, double* __restrict__ q)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    if (j1 <= j0) return;
    const double uni = Qb[b] / (j1 - j0);
    double mean = 0.0;
    if (warm) {
        double s = 0.0;
        for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) s += q[j];
        mean = block_sum(s, sh) / (j1 - j0);
    }
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) q[j] = warm ? (q[j] - mean + uni) : uni;
}

__global__ void k_copy(int n, const double* __restrict__ in, double* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i];
}

// g = P(r.E0 - psi0), p = g; per-body partials of |g|^2 and of the reference norm
__global__ void __launch_bounds__(BT)
k_resid_init(const int* __restrict__ off, const double* __restrict__ rx, const double* __restrict__ ry, const double* __restrict__ rz,
             double e0x, double e0y, double e0z, const double* __restrict__ psi0, double* __restrict__ rhs, double* __restrict__ g,
             double* __restrict__ p, double* __restrict__ part_gg, double* __restrict__ part_ref)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    if (j1 <= j0) { if (threadIdx.x == 0) { part_gg[b] = 0; part_ref[b] = 0; } return; }
    double s = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) s += psi0[j];
    const double mean = block_sum(s, sh) / (j1 - j0);
    double gg = 0.0, rf = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double re = rx[j] * e0x + ry[j] * e0y + rz[j] * e0z;  // sum_j r_ij = 0, so P(r.E0) = r.E0
        const double pc = psi0[j] - mean;
        const double v = re - pc;
        rhs[j] = re; g[j] = v; p[j] = v;
        gg += v * v; rf += re * re + pc * pc;
    }
    gg = block_sum(gg, sh);
    rf = block_sum(rf, sh);
    if (threadIdx.x == 0) { part_gg[b] = gg; part_ref[b] = rf; }
}

// ap = P t ; partial of p.ap
__global__ void __launch_bounds__(BT)
k_proj_dot(const int* __restrict__ off, const double* __restrict__ t, const double* __restrict__ p, double* __restrict__ ap,
           double* __restrict__ part)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    if (j1 <= j0) { if (threadIdx.x == 0) part[b] = 0; return; }
    double s = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) s += t[j];
    const double mean = block_sum(s, sh) / (j1 - j0);
    double d = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double v = t[j] - mean;
        ap[j] = v;
        d += p[j] * v;
    }
    d = block_sum(d, sh);
    if (threadIdx.x == 0) part[b] = d;
}

// alpha = (g.z)/pAp ; q += alpha p ; g -= alpha ap ; psi += alpha t ; partial of |g|^2
__global__ void __launch_bounds__(BT)
k_cg_update(const int* __restrict__ off, const double* __restrict__ sc_gg, const double* __restrict__ sc_pap,
            const double* __restrict__ p, const double* __restrict__ ap, const double* __restrict__ t, double* __restrict__ q,
            double* __restrict__ g, double* __restrict__ psi, double* __restrict__ part)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    const double pap = sc_pap[0];
    const double alpha = (pap != 0.0) ? sc_gg[0] / pap : 0.0;
    double gg = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        q[j] += alpha * p[j];
        psi[j] += alpha * t[j];
        const double v = g[j] - alpha * ap[j];
        g[j] = v;
        gg += v * v;
    }
    gg = block_sum(gg, sh);
    if (threadIdx.x == 0) part[b] = gg;
}

// beta = rz_new/rz_old (0 on the first call) ; p = z + beta p with z = g (no preconditioner) or
// z = z_raw - <z_raw>_body (block-Jacobi, precond.cu)
__global__ void k_cg_pupdate(int n, const double* __restrict__ sc_old, const double* __restrict__ sc_new, const double* __restrict__ g,
                             const double* __restrict__ zraw, const double* __restrict__ zmean, const int* __restrict__ body_of,
                             double* __restrict__ p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double beta = 0.0;
    if (sc_old) {
        const double o = sc_old[0];
        beta = (o != 0.0) ? sc_new[0] / o : 0.0;
    }
    const double z = zraw ? zraw[i] - zmean[body_of[i]] : g[i];
    p[i] = sc_old ? z + beta * p[i] : z;
}

// per body: mean of z_raw and the partial of g.z (g has zero mean per body, so g.z = g.z_raw)
__global__ void __launch_bounds__(BT)
k_pc_dot(const int* __restrict__ off, const double* __restrict__ zraw, const double* __restrict__ g, double* __restrict__ zmean,
         double* __restrict__ part)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    double s = 0.0, d = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) { const double z = zraw[j]; s += z; d += g[j] * z; }
    s = block_sum(s, sh);
    d = block_sum(d, sh);
    if (threadIdx.x == 0) { zmean[b] = (j1 > j0) ? s / (j1 - j0) : 0.0; part[b] = d; }
}

// Phi_i = <psi_ij - r_ij.E0>_i = <psi_ij>_i
__global__ void __launch_bounds__(BT)
k_body_mean(const int* __restrict__ off, const double* __restrict__ v, double* __restrict__ out)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    double s = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) s += v[j];
    s = block_sum(s, sh);
    if (threadIdx.x == 0) out[b] = (j1 > j0) ? s / (j1 - j0) : 0.0;
}

int solve_cg(pce_ctx* c, const double* Q_body, const double* q_ion, const double E0[3], int warm, double* q, double* Phi,
             pce_solve_info* info)
{
    const int nb = c->Nbody, nbead = c->Nbead, N = c->N;
    pce_solve_info inf = {0, 0, 0.0, 1};
    // 1. starting charges
    if (nb > 0) {
        PassTimer t(c, PASS_KRYLOV);
        k_init_q<<<nb, BT, 0, c->st>>>(c->body_off, Q_body, warm, q);
        c->launches++;
    }
    if (c->Nion > 0) {
        if (!q_ion) { c->err = "q_ion is NULL but the system has ions"; return PCE_EINVAL; }
        k_copy<<<cdiv(c->Nion, 256), 256, 0, c->st>>>(c->Nion, q_ion, q + nbead);
        c->launches++;
    }
    PCE_CUDA(c, cudaGetLastError());
    if (nb == 0 || nbead == 0) {
        if (info) *info = inf;
        return PCE_OK;
    }
    // 2. potentials of the starting charges at every bead (ions included as sources): all sources, bead targets
    int rc = op_evaluate_at_beads(c, q, c->ev_psi);
    if (rc) return rc;
    inf.matvecs = 1;
    const int maxit = c->p.max_iter;
    // device scalars: [0] = ref^2, [1] = |g_0|^2; iteration it: g.z at 2+3it, p.Ap at 3+3it, |g_{it+1}|^2 at 4+3it
    double* sc = c->cg_scal;
    double* part = c->cg_scal + 3 * (maxit + 2) + 2;  // [nb] partials
    double* part2 = part + nb;
    const bool pc = c->pc_on;
    const double* zraw = pc ? c->cg_z : nullptr;
    double* cur_rz = pc ? sc + 2 : sc + 1;
    {
        PassTimer t(c, PASS_KRYLOV);
        k_copy<<<cdiv(nbead, 256), 256, 0, c->st>>>(nbead, c->ev_psi, c->cg_psi);
        k_resid_init<<<nb, BT, 0, c->st>>>(c->body_off, c->rx, c->ry, c->rz, E0[0], E0[1], E0[2], c->ev_psi, c->cg_rhs, c->cg_g,
                                         c->cg_p, part, part2);
        c->launches += 2;
        if ((rc = sum_to(c, part, nb, sc + 1))) return rc;
        if ((rc = sum_to(c, part2, nb, sc + 0))) return rc;
        if (pc) {
            if ((rc = precond_apply(c, c->cg_g, c->cg_z))) return rc;
            k_pc_dot<<<nb, BT, 0, c->st>>>(c->body_off, c->cg_z, c->cg_g, c->pc_mean, part);
            c->launches++;
            if ((rc = sum_to(c, part, nb, cur_rz))) return rc;
            k_cg_pupdate<<<cdiv(nbead, 256), 256, 0, c->st>>>(nbead, nullptr, nullptr, c->cg_g, zraw, c->pc_mean, c->body_of, c->cg_p);
            c->launches++;
        }
    }
    double ref2 = 0.0, gg = 0.0;
    PCE_CUDA(c, cudaMemcpyAsync(&ref2, sc + 0, sizeof(double), cudaMemcpyDeviceToHost, c->st));
    PCE_CUDA(c, cudaMemcpyAsync(&gg, sc + 1, sizeof(double), cudaMemcpyDeviceToHost, c->st));
    PCE_CUDA(c, cudaStreamSynchronize(c->st));
    // Scale of the data: (|P r.E0|^2 + |P psi0|^2)^(1/2) with psi0 the potential of the uniform starting charges and the
    // ions.  After a warm start psi0 is already nearly equipotential and that norm collapses, so the scale of the last cold
    // solve of this system is kept and used whenever it is larger.
    double ref = (ref2 > 0.0) ? sqrt(ref2) : 1.0;
    if (!warm) c->cg_ref_cold = ref;
    else if (c->cg_ref_cold > ref) ref = c->cg_ref_cold;
    const double tol = c->p.tol_solver;
    int it = 0;
    inf.rel_resid = sqrt(gg) / ref;
    while (inf.rel_resid > tol && it < maxit) {
        double* s_pap = sc + 3 + 3 * it;
        double* s_gn = sc + 4 + 3 * it;
        double* next_rz = pc ? sc + 2 + 3 * (it + 1) : s_gn;
        if ((rc = op_matvec_bead(c, c->cg_p, c->cg_t))) return rc;
        inf.matvecs++;
        {
            PassTimer t(c, PASS_KRYLOV);
            k_proj_dot<<<nb, BT, 0, c->st>>>(c->body_off, c->cg_t, c->cg_p, c->cg_ap, part);
            c->launches++;
            if ((rc = sum_to(c, part, nb, s_pap))) return rc;
            k_cg_update<<<nb, BT, 0, c->st>>>(c->body_off, cur_rz, s_pap, c->cg_p, c->cg_ap, c->cg_t, q, c->cg_g, c->cg_psi, part);
            c->launches++;
            if ((rc = sum_to(c, part, nb, s_gn))) return rc;
            PCE_CUDA(c, cudaMemcpyAsync(&gg, s_gn, sizeof(double), cudaMemcpyDeviceToHost, c->st));
            if (pc) {
                if ((rc = precond_apply(c, c->cg_g, c->cg_z))) return rc;
                k_pc_dot<<<nb, BT, 0, c->st>>>(c->body_off, c->cg_z, c->cg_g, c->pc_mean, part);
                c->launches++;
                if ((rc = sum_to(c, part, nb, next_rz))) return rc;
            }
            k_cg_pupdate<<<cdiv(nbead, 256), 256, 0, c->st>>>(nbead, cur_rz, next_rz, c->cg_g, zraw, c->pc_mean, c->body_of, c->cg_p);
            c->launches++;
        }
        PCE_CUDA(c, cudaStreamSynchronize(c->st));
        cur_rz = next_rz;
        ++it;
        inf.rel_resid = sqrt(gg) / ref;
        if (!(gg == gg)) { c->err = "NaN in the Krylov residual"; return PCE_ECUDA; }
    }
    inf.iters = it;
    inf.converged = (inf.rel_resid <= tol) ? 1 : 0;
    {
        PassTimer t(c, PASS_KRYLOV);
        k_body_mean<<<nb, BT, 0, c->st>>>(c->body_off, c->cg_psi, Phi);
        c->launches++;
    }
    PCE_CUDA(c, cudaGetLastError());
    if (info) *info = inf;
    (void)N;
    return inf.converged ? PCE_OK : PCE_ENOCONV;
}

// ---------------------------------------------------------------- forces, torques, moments, energies
__global__ void k_force(int n, const double* __restrict__ q, const double* __restrict__ ex, const double* __restrict__ ey,
                        const double* __restrict__ ez, double e0x, double e0y, double e0z, double* __restrict__ fx,
                        double* __restrict__ fy, double* __restrict__ fz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double qi = q[i];
    fx[i] = qi * (e0x + ex[i]); fy[i] = qi * (e0y + ey[i]); fz[i] = qi * (e0z + ez[i]);  // eq. 17 = eq. 58
}

__global__ void __launch_bounds__(BT)
k_body_moments(int nb, const int* __restrict__ off, const double* __restrict__ q, const double* __restrict__ psi,
               const double* __restrict__ fx, const double* __restrict__ fy, const double* __restrict__ fz,
               const double* __restrict__ rx, const double* __restrict__ ry, const double* __restrict__ rz,
               const double* __restrict__ X, const double* __restrict__ Y, const double* __restrict__ Z, double e0x, double e0y,
               double e0z, double* __restrict__ F, double* __restrict__ T, double* __restrict__ S, double* __restrict__ U)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    double a[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};  // F(3) T(3) S(3) Q sum(psi - r.E0)
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double f0 = fx[j], f1 = fy[j], f2 = fz[j], r0 = rx[j], r1 = ry[j], r2 = rz[j], qj = q[j];
        a[0] += f0; a[1] += f1; a[2] += f2;
        a[3] += r1 * f2 - r2 * f1; a[4] += r2 * f0 - r0 * f2; a[5] += r0 * f1 - r1 * f0;  // eq. 18
        a[6] += r0 * qj; a[7] += r1 * qj; a[8] += r2 * qj;                                // eq. 14
        a[9] += qj;
        a[10] += psi[j] - (r0 * e0x + r1 * e0y + r2 * e0z);
    }
#pragma unroll
    for (int k = 0; k < 11; ++k) a[k] = block_sum(a[k], sh);
    if (threadIdx.x == 0) {
        if (F) { F[b] = a[0]; F[nb + b] = a[1]; F[2 * nb + b] = a[2]; }
        if (T) { T[b] = a[3]; T[nb + b] = a[4]; T[2 * nb + b] = a[5]; }
        if (S) { S[b] = a[6]; S[nb + b] = a[7]; S[2 * nb + b] = a[8]; }
        const double Phi = (j1 > j0) ? a[10] / (j1 - j0) : 0.0;
        const double Psi = Phi - (X[b] * e0x + Y[b] * e0y + Z[b] * e0z);  // Psi_0,i = -X_i.E0
        U[b] = 0.5 * (a[9] * Psi - (a[6] * e0x + a[7] * e0y + a[8] * e0z));  // eq. 16, first line
    }
}

// per-particle energy terms: e1 = q psi / 2, e2 = q x.E0 with x = X_i + r_ij (beads) or the ion position
__global__ void k_energy_terms(int n, int nbead, const int* __restrict__ body_of, const double* __restrict__ q,
                               const double* __restrict__ psi, const double* __restrict__ x, const double* __restrict__ y,
                               const double* __restrict__ z, const double* __restrict__ rx, const double* __restrict__ ry,
                               const double* __restrict__ rz, const double* __restrict__ X, const double* __restrict__ Y,
                               const double* __restrict__ Z, double e0x, double e0y, double e0z, double* __restrict__ e1,
                               double* __restrict__ e2, double* __restrict__ U_ion)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double px, py, pz;
    if (i < nbead) {
        const int b = body_of[i];
        px = X[b] + rx[i]; py = Y[b] + ry[i]; pz = Z[b] + rz[i];
    } else {
        px = x[i]; py = y[i]; pz = z[i];
    }
    const double xe = px * e0x + py * e0y + pz * e0z;
    e1[i] = 0.5 * q[i] * psi[i];
    e2[i] = q[i] * xe;
    if (i >= nbead) U_ion[i - nbead] = 0.5 * q[i] * (psi[i] - xe);
}

__global__ void k_energy_final(const double* __restrict__ s, double* __restrict__ U_tot)
{
    // s[0] = sum U_i (bodies + ions), s[1] = U_MM, s[2] = sum q x.E0
    U_tot[0] = s[0]; U_tot[1] = s[1] - s[2]; U_tot[2] = s[1];
}

int forces_all(pce_ctx* c, const double* q, const double E0[3], double* fx, double* fy, double* fz, double* F, double* T, double* S,
               double* U_body, double* U_tot, double* psi_out)
{
    const int N = c->N, nb = c->Nbody, nbead = c->Nbead;
    int rc = op_evaluate(c, q, c->ev_psi, c->ev_ex, c->ev_ey, c->ev_ez);
    if (rc) return rc;
    PassTimer t(c, PASS_OTHER);
    // bead forces go to the caller's arrays if given, else to scratch (w_k* are free after the evaluation)
    double* gx = fx ? fx : c->w_kx;
    double* gy = fy ? fy : c->w_ky;
    double* gz = fz ? fz : c->w_kz;
    k_force<<<cdiv(N, 256), 256, 0, c->st>>>(N, q, c->ev_ex, c->ev_ey, c->ev_ez, E0[0], E0[1], E0[2], gx, gy, gz);
    c->launches++;
    double* Ub = U_body ? U_body : c->w_real;  // [nb + Nion]
    if (nb > 0) {
        k_body_moments<<<nb, BT, 0, c->st>>>(nb, c->body_off, q, c->ev_psi, gx, gy, gz, c->rx, c->ry, c->rz, c->X, c->Y, c->Z, E0[0],
                                           E0[1], E0[2], F, T, S, Ub);
        c->launches++;
    }
    if (U_tot || U_body) {
        double* e1 = c->w_ex;
        double* e2 = c->w_ey;
        k_energy_terms<<<cdiv(N, 256), 256, 0, c->st>>>(N, nbead, c->body_of, q, c->ev_psi, c->x, c->y, c->z, c->rx, c->ry, c->rz, c->X,
                                                       c->Y, c->Z, E0[0], E0[1], E0[2], e1, e2, Ub + nb);
        c->launches++;
        if (U_tot) {
            if ((rc = sum_vector(c, Ub, nb + c->Nion, c->scal + 4))) return rc;
            if ((rc = sum_vector(c, e1, N, c->scal + 5))) return rc;
            if ((rc = sum_vector(c, e2, N, c->scal + 6))) return rc;
            k_energy_final<<<1, 1, 0, c->st>>>(c->scal + 4, U_tot);
            c->launches++;
        }
    }
    if (psi_out) {
        k_copy<<<cdiv(N, 256), 256, 0, c->st>>>(N, c->ev_psi, psi_out);
        c->launches++;
    }
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
