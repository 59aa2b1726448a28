// krylov.cu -- rigid-body bookkeeping (Sigma of eq. 13 / eq. 52 as contiguous
// bead ranges), the on-device conjugate-gradient solve of the induced-charge
// saddle-point system eq. 13 in its per-body-mean-projected SPD
// form, and the moments / forces / torques / energies of eqs. 14, 16-18
// (PAPER.md:137-163).  All reductions have a fixed order (deterministic).
#include "pce_internal.h"

#include <cstdlib>

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

// caller-supplied centres (pce_set_centres): r_ij = minimum image of x_ij - X_i
__global__ void k_rel_to_centres(int nbead, const int* __restrict__ body_of, const double* __restrict__ x, const double* __restrict__ y,
                                 const double* __restrict__ z, const double* __restrict__ X, const double* __restrict__ Y,
                                 const double* __restrict__ Z, double Lx, double Ly, double Lz, double* __restrict__ rx,
                                 double* __restrict__ ry, double* __restrict__ rz)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nbead) return;
    const int b = body_of[j];
    rx[j] = min_img(x[j] - X[b], Lx); ry[j] = min_img(y[j] - Y[b], Ly); rz[j] = min_img(z[j] - Z[b], Lz);
}

int bodies_set_centres(pce_ctx* c, const double* X, const double* Y, const double* Z)
{
    if (c->Nbody == 0) return PCE_OK;
    PCE_CUDA(c, cudaMemcpyAsync(c->X, X, (size_t)c->Nbody * 8, cudaMemcpyDeviceToDevice, c->st));
    PCE_CUDA(c, cudaMemcpyAsync(c->Y, Y, (size_t)c->Nbody * 8, cudaMemcpyDeviceToDevice, c->st));
    PCE_CUDA(c, cudaMemcpyAsync(c->Z, Z, (size_t)c->Nbody * 8, cudaMemcpyDeviceToDevice, c->st));
    k_rel_to_centres<<<cdiv(c->Nbead, 256), 256, 0, c->st>>>(c->Nbead, c->body_of, c->x, c->y, c->z, c->X, c->Y, c->Z, c->p.L[0], c->p.L[1],
                                                            c->p.L[2], c->rx, c->ry, c->rz);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// ---------------------------------------------------------------- Krylov solve, whole iteration on the device
// Conjugate gradients for eq. 13 with the ions eliminated (one-bead bodies of fixed charge):
//     P M_bb P q = P b  on  Sigma q = Q,   P = I - Sigma^T (Sigma Sigma^T)^-1 Sigma  (subtract the per-body mean),
// preconditioned by the rigid-body blocks of precond.cu; with project = 0 the same loop solves the plain SPD system
// M_bb q = b (columns of the grand capacitance tensor, eq. 15).  All step lengths, the stopping test and the iteration
// count live in CgState on the device; every sum is a per-block partial followed by a fixed-order sum in the block that
// arrives last (deterministic, no extra launch).  One iteration is 5 own kernels + the operator and is replayed as a CUDA
// graph; once converged every kernel of a replay returns at once.  The host never synchronises inside the loop: it
// watches CgHostStatus (pinned, mapped) and keeps `depth` iterations in flight.

// true (for the whole block) in the block that arrives last; the counter is left at 0 for the next use
__device__ __forceinline__ bool last_block_done(unsigned* counter, unsigned nblocks)
{
    __shared__ bool last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(counter, 1u);
        last = (t == nblocks - 1);
        if (last) *counter = 0u;
    }
    __syncthreads();
    if (last) __threadfence();
    return last;
}

__device__ __forceinline__ double fixed_sum(const double* part, int n, double* sh)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) v += part[i];
    return block_sum(v, sh);
}

__device__ __forceinline__ void report(const CgState* st, CgHostStatus* hs)
{
    hs->gg = st->gg; hs->ref = st->ref;
    __threadfence_system();
    hs->it = st->it; hs->done = st->done;
    __threadfence_system();
}

// initial charges: beads Q_i/N_i (or the caller's guess re-centred so that sum_j q_ij = Q_i)
__global__ void __launch_bounds__(BT)
k_init_q(const int* __restrict__ off, const double* __restrict__ Qb, int warm, const double* __restrict__ q_in, double* __restrict__ q)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    if (j1 <= j0) return;
    const double uni = Qb[b] / (j1 - j0);
    double mean = 0.0;
    if (warm) {
        double s = 0.0;
        for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) s += q_in[j];
        mean = block_sum(s, sh) / (j1 - j0);
    }
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) q[j] = warm ? (q_in[j] - mean + uni) : uni;
}

__global__ void k_copy(int n, const double* __restrict__ in, double* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i];
}

// g = P(r.E0 - psi0) (one CTA per body); the last block sets up the solver state: |g|^2, the residual scale
//   ref^2 = |P r.E0|^2 + |P psi0|^2 + 1e-4 |psi0|^2
// (psi0 = potential of the starting charges and the ions; the unprojected term keeps the scale meaningful when psi0 is
// already nearly equipotential, e.g. an isolated charged body without field), warm starts keep the scale of the last cold solve.
__global__ void __launch_bounds__(BT)
k_resid_init(int nb, const int* __restrict__ off, const double* __restrict__ rx, const double* __restrict__ ry, const double* __restrict__ rz,
             double e0x, double e0y, double e0z, const double* __restrict__ psi0, double* __restrict__ g, double* __restrict__ part,
             CgState* __restrict__ st, CgHostStatus* __restrict__ hs, int warm, int have_pc, double tol, int maxit)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    // per-body means of psi0 and of r.E0 (the latter is 0 for bead-mean centres, not for caller-supplied ones: pce_set_centres)
    double s = 0.0, sr = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) { s += psi0[j]; sr += rx[j] * e0x + ry[j] * e0y + rz[j] * e0z; }
    const double mean = (j1 > j0) ? block_sum(s, sh) / (j1 - j0) : 0.0;
    const double mean_re = (j1 > j0) ? block_sum(sr, sh) / (j1 - j0) : 0.0;
    double gg = 0.0, rf = 0.0, pp = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double re = rx[j] * e0x + ry[j] * e0y + rz[j] * e0z - mean_re;  // P(r.E0)
        const double p0 = psi0[j], pc = p0 - mean;
        const double v = re - pc;
        g[j] = v;
        gg += v * v; rf += re * re + pc * pc; pp += p0 * p0;
    }
    gg = block_sum(gg, sh);
    rf = block_sum(rf, sh);
    pp = block_sum(pp, sh);
    if (threadIdx.x == 0) { part[b] = gg; part[nb + b] = rf; part[2 * nb + b] = pp; }
    if (!last_block_done(&st->cnt[0], gridDim.x)) return;
    const double tgg = fixed_sum(part, nb, sh), trf = fixed_sum(part + nb, nb, sh), tpp = fixed_sum(part + 2 * nb, nb, sh);
    if (threadIdx.x == 0) {
        const double r2 = trf + 1e-4 * tpp;
        double ref = (r2 > 0.0) ? sqrt(r2) : 1.0;
        if (!warm) st->ref_cold = ref;
        else if (st->ref_cold > ref) ref = st->ref_cold;
        st->ref = ref; st->gg = tgg; st->tol = tol; st->maxit = maxit; st->it = 0; st->project = 1; st->psum = 0.0; st->pap = 0.0;
        st->rz[0] = tgg; st->rz[1] = tgg;
        st->done = (!(sqrt(tgg) > tol * ref) || maxit <= 0) ? 1 : 0;   // NaN counts as done (reported as not converged)
        if (!have_pc || st->done) report(st, hs);
    }
}

// save (restore = 0) / put back (restore = 1) the residual scale of the last cold-start solve around internal solves
__global__ void k_ref_cold_keep(CgState* __restrict__ st, int restore)
{
    if (restore) st->ref_cold = st->ref_saved;
    else st->ref_saved = st->ref_cold;
}

// plain system M q = b from q = 0: g = b; ref = |b|
__global__ void __launch_bounds__(BT)
k_resid_init_plain(int n, const double* __restrict__ b, double* __restrict__ g, double* __restrict__ q, double* __restrict__ psi,
                   double* __restrict__ part, CgState* __restrict__ st, CgHostStatus* __restrict__ hs, int have_pc, double tol, int maxit)
{
    __shared__ double sh[32];
    double gg = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double v = b[i];
        g[i] = v; q[i] = 0.0; psi[i] = 0.0;
        gg += v * v;
    }
    gg = block_sum(gg, sh);
    if (threadIdx.x == 0) part[blockIdx.x] = gg;
    if (!last_block_done(&st->cnt[0], gridDim.x)) return;
    const double tgg = fixed_sum(part, gridDim.x, sh);
    if (threadIdx.x == 0) {
        st->ref = (tgg > 0.0) ? sqrt(tgg) : 1.0;
        st->gg = tgg; st->tol = tol; st->maxit = maxit; st->it = 0; st->project = 0; st->psum = 0.0; st->pap = 0.0;
        st->rz[0] = tgg; st->rz[1] = tgg;
        st->done = (!(sqrt(tgg) > tol * st->ref) || maxit <= 0) ? 1 : 0;
        if (!have_pc || st->done) report(st, hs);
    }
}

// z = preconditioned residual, per body (one CTA):  project: z_raw - <z_raw>_body;  plain: z_raw + u (u.g)/(1.u)  (A^-1 from its
// projected part B, precond.cu);  without a preconditioner z = g.  Partial of g.z; the last block stores g.z at rz[it & 1].
__global__ void __launch_bounds__(BT)
k_pc_dot(int nb, const int* __restrict__ off, double* __restrict__ zraw, const double* __restrict__ g, const double* __restrict__ u,
         const double* __restrict__ inv_s, double* __restrict__ zmean, double* __restrict__ part, CgState* __restrict__ st,
         CgHostStatus* __restrict__ hs, int report_init)
{
    if (st->done) return;
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    const int project = st->project;
    double s = 0.0, d = 0.0, ug = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double z = zraw[j], gj = g[j];
        s += z; d += gj * z; ug += u[j] * gj;
    }
    s = block_sum(s, sh);
    d = block_sum(d, sh);
    if (project) {
        if (threadIdx.x == 0) zmean[b] = (j1 > j0) ? s / (j1 - j0) : 0.0;  // g has zero mean per body: g.z = g.z_raw
    } else {
        ug = block_sum(ug, sh);
        const double cfac = ug * inv_s[b];  // 0 for bodies without a dense block
        for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) zraw[j] += cfac * u[j];
        d += cfac * ug;
        if (threadIdx.x == 0) zmean[b] = 0.0;
    }
    if (threadIdx.x == 0) part[b] = d;
    if (!last_block_done(&st->cnt[1], gridDim.x)) return;
    const double t = fixed_sum(part, nb, sh);
    if (threadIdx.x == 0) {
        st->rz[st->it & 1] = t;
        if (report_init) report(st, hs);
    }
}

// p = z + beta p, beta = rz_new / rz_old (p = z in the first iteration), written in caller order and scattered into the two
// sorted orders the operator reads (real-space cells, mesh bins); partial of sum(p) for the k = 0 constant
__global__ void __launch_bounds__(256)
k_pupdate(int n, const double* __restrict__ g, const double* __restrict__ zraw, const double* __restrict__ zmean,
          const int* __restrict__ body_of, const int* __restrict__ inv_r, const int* __restrict__ inv_w, double* __restrict__ p,
          double* __restrict__ qs_r, double* __restrict__ qs_w, int qs_w_stride, double* __restrict__ part, CgState* __restrict__ st)
{
    if (st->done) return;
    __shared__ double sh[32];
    const int it = st->it;
    double beta = 0.0;
    if (it > 0) {
        const double o = st->rz[(it + 1) & 1];
        beta = (o != 0.0) ? st->rz[it & 1] / o : 0.0;
    }
    double ps = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double z = zraw ? zraw[i] - zmean[body_of[i]] : g[i];
        const double v = (it > 0) ? z + beta * p[i] : z;
        p[i] = v;
        qs_r[inv_r[i]] = v;
        qs_w[(size_t)inv_w[i] * qs_w_stride] = v;
        ps += v;
    }
    ps = block_sum(ps, sh);
    if (threadIdx.x == 0) part[blockIdx.x] = ps;
    if (!last_block_done(&st->cnt[2], gridDim.x)) return;
    const double t = fixed_sum(part, gridDim.x, sh);
    if (threadIdx.x == 0) st->psum = t;
}

// t = M p assembled from the sorted real- and wave-space parts (step "a8", reading A1), ap = P t (or t), partial of p.ap
__global__ void __launch_bounds__(BT)
k_proj_dot(int nb, const int* __restrict__ off, const int* __restrict__ inv_r, const int* __restrict__ inv_w, const double* __restrict__ re,
           const double* __restrict__ wa, double kconst, const double* __restrict__ p, double* __restrict__ t, double* __restrict__ ap,
           double* __restrict__ part, CgState* __restrict__ st)
{
    if (st->done) return;
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    const double shift = kconst * st->psum;
    double s = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double v = re[inv_r[j]] + wa[inv_w[j]] - shift;
        t[j] = v;
        s += v;
    }
    const double mean = (st->project && j1 > j0) ? block_sum(s, sh) / (j1 - j0) : 0.0;
    double d = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double v = t[j] - mean;
        ap[j] = v;
        d += p[j] * v;
    }
    d = block_sum(d, sh);
    if (threadIdx.x == 0) part[b] = d;
    if (!last_block_done(&st->cnt[3], gridDim.x)) return;
    const double tt = fixed_sum(part, nb, sh);
    if (threadIdx.x == 0) st->pap = tt;
}

// alpha = (g.z)/(p.Ap); q += alpha p; psi += alpha t; g -= alpha ap; the last block: |g|^2, iteration count, stopping test
__global__ void __launch_bounds__(BT)
k_cg_update(int nb, const int* __restrict__ off, const double* __restrict__ p, const double* __restrict__ ap, const double* __restrict__ t,
            double* __restrict__ q, double* __restrict__ g, double* __restrict__ psi, double* __restrict__ part, CgState* __restrict__ st,
            CgHostStatus* __restrict__ hs, int have_pc)
{
    if (st->done) return;
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    const int it = st->it;
    const double pap = st->pap;
    const double alpha = (pap != 0.0) ? st->rz[it & 1] / pap : 0.0;
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
    if (!last_block_done(&st->cnt[4], gridDim.x)) return;
    const double tg = fixed_sum(part, nb, sh);
    if (threadIdx.x == 0) {
        st->gg = tg;
        st->it = it + 1;
        if (!have_pc) st->rz[(it + 1) & 1] = tg;
        if (!(sqrt(tg) > st->tol * st->ref) || it + 1 >= st->maxit) st->done = 1;
        report(st, hs);
    }
}

// Phi_i = <psi_ij - r_ij.E0>_i  (= <psi_ij>_i for bead-mean centres)
__global__ void __launch_bounds__(BT)
k_body_mean(const int* __restrict__ off, const double* __restrict__ v, const double* __restrict__ rx, const double* __restrict__ ry,
            const double* __restrict__ rz, double e0x, double e0y, double e0z, double* __restrict__ out)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    double s = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) s += v[j] - (rx[j] * e0x + ry[j] * e0y + rz[j] * e0z);
    s = block_sum(s, sh);
    if (threadIdx.x == 0) out[b] = (j1 > j0) ? s / (j1 - j0) : 0.0;
}

static int pupdate_blocks(const pce_ctx* c) { int b = cdiv(c->Nbead, 256 * 4); return b < 1 ? 1 : (b > 1024 ? 1024 : b); }

static int krylov_alloc(pce_ctx* c)
{
    if (c->cg_state) return PCE_OK;
    PCE_CUDA(c, cudaMalloc(&c->cg_state, sizeof(CgState)));
    PCE_CUDA(c, cudaMemset(c->cg_state, 0, sizeof(CgState)));
    PCE_CUDA(c, cudaHostAlloc(&c->cg_host, sizeof(CgHostStatus), cudaHostAllocMapped));
    PCE_CUDA(c, cudaHostGetDevicePointer(&c->cg_host_dev, c->cg_host, 0));
    c->cg_host->it = 0; c->cg_host->done = 0; c->cg_host->gg = 0.0; c->cg_host->ref = 1.0;
    return PCE_OK;
}

// The captured iteration bakes in device pointers (csr_col / csr_val, gather_part, the hit and pair lists), sizes (nnz, n_items,
// n_pairs) and grid dimensions, all of which change with the positions or with a reallocation: whoever changes one of them calls
// this, and the next solve captures the iteration again (updating the instantiated graph in place where the topology is unchanged).
void krylov_invalidate_graph(pce_ctx* c) { c->cg_graph_stale = true; }

static void destroy_graph(pce_ctx* c)
{
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }
    c->cg_graph_stale = false;
}

void krylov_free(pce_ctx* c)
{
    destroy_graph(c);
    cudaFree(c->cg_state);
    if (c->cg_host) cudaFreeHost(c->cg_host);
    c->cg_state = nullptr; c->cg_host = nullptr; c->cg_host_dev = nullptr; c->cg_graph_failed = false;
}

// the preconditioned residual and g.z for the current g (also used once before the loop)
static int enqueue_precond(pce_ctx* c, int report_init)
{
    int rc = precond_apply(c, c->cg_g, c->cg_z);
    if (rc) return rc;
    k_pc_dot<<<c->Nbody, BT, 0, c->st>>>(c->Nbody, c->body_off, c->cg_z, c->cg_g, c->pc_u, c->pc_invs, c->pc_mean, c->cg_part, c->cg_state,
                                        c->cg_host_dev, report_init);
    c->launches++;
    return PCE_OK;
}

// one iteration: search direction, operator, step.  Every kernel returns at once when the state says "done".
static int enqueue_iteration(pce_ctx* c)
{
    const int nb = c->Nbody, n = c->Nbead;
    const bool pc = c->pc_on;
    int rc;
    c->skip_flag = &c->cg_state->done;
    {
        PassTimer t(c, PASS_KRYLOV);
        k_pupdate<<<pupdate_blocks(c), 256, 0, c->st>>>(n, c->cg_g, pc ? c->cg_z : nullptr, c->pc_mean, c->body_of, c->bead.inv, c->wmv->inv,
                                                        c->cg_p, c->bead.qs, c->use_cols ? c->wmv->qs_cols : c->wmv->qs, c->use_cols ? HITREC_Q_STRIDE : 1, c->cg_part, c->cg_state);
        c->launches++;
    }
    rc = op_matvec_bead_sorted(c);
    if (!rc) {
        PassTimer t(c, PASS_KRYLOV);
        k_proj_dot<<<nb, BT, 0, c->st>>>(nb, c->body_off, c->bead.inv, c->wmv->inv, c->w_real, c->w_wave, c->kconst, c->cg_p, c->cg_t, c->cg_ap,
                                        c->cg_part, c->cg_state);
        k_cg_update<<<nb, BT, 0, c->st>>>(nb, c->body_off, c->cg_p, c->cg_ap, c->cg_t, c->cg_q, c->cg_g, c->cg_psi, c->cg_part, c->cg_state,
                                         c->cg_host_dev, pc ? 1 : 0);
        c->launches += 2;
        if (pc) rc = enqueue_precond(c, 0);
    }
    c->skip_flag = nullptr;
    if (rc) return rc;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

static bool graphs_enabled()
{
    static int on = -1;
    if (on < 0) { const char* e = getenv("PCE_NO_GRAPH"); on = (e && e[0] == '1') ? 0 : 1; }
    return on == 1;
}

// capture one iteration into a graph (again after every krylov_invalidate_graph; arrays it touches are owned by the context).
// The legacy default stream cannot be captured (cudaStreamBeginCapture fails on it): a context created on it runs plain launches.
static int capture_iteration(pce_ctx* c)
{
    cudaGraph_t g = nullptr;
    const long long l0 = c->launches;
    c->cg_graph_stale = false;
    if (cudaStreamBeginCapture(c->st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); destroy_graph(c); c->cg_graph_failed = true; return PCE_OK; }
    const int rc = enqueue_iteration(c);
    const cudaError_t e = cudaStreamEndCapture(c->st, &g);
    c->cg_graph_launches = c->launches - l0;
    c->launches = l0;
    if (rc != PCE_OK || e != cudaSuccess || !g) {
        cudaGetLastError();
        if (g) cudaGraphDestroy(g);
        destroy_graph(c);
        c->cg_graph_failed = true;  // fall back to plain launches
        return PCE_OK;
    }
    if (c->cg_graph) {  // same topology, new arguments: update in place; otherwise instantiate afresh
        cudaGraphExecUpdateResultInfo upd;
        if (cudaGraphExecUpdate(c->cg_graph, g, &upd) != cudaSuccess) { cudaGetLastError(); destroy_graph(c); }
    }
    if (!c->cg_graph && cudaGraphInstantiate(&c->cg_graph, g, 0) != cudaSuccess) { cudaGetLastError(); c->cg_graph = nullptr; c->cg_graph_failed = true; }
    cudaGraphDestroy(g);
    return PCE_OK;
}

// wait (without touching the stream) until the device reports iteration `want` complete or the solve done
static int wait_progress(pce_ctx* c, int want)
{
    volatile CgHostStatus* hs = c->cg_host;
    long spins = 0;
    while (hs->it < want && !hs->done) {
        if ((++spins & 1023) == 0) {
            const cudaError_t e = cudaStreamQuery(c->st);
            if (e == cudaSuccess) {  // nothing left in the stream
                if (hs->it < want && !hs->done) { c->err = "Krylov solve: the device stopped reporting progress"; return PCE_ECUDA; }
            } else if (e != cudaErrorNotReady) {
                c->err = std::string("Krylov solve: ") + cudaGetErrorString(e);
                return PCE_ECUDA;
            }
        }
    }
    return PCE_OK;
}

// the loop shared by both systems; the state has been initialised on the device (it = 0, done, rz[0])
static int run_iterations(pce_ctx* c, pce_solve_info* inf)
{
    const int maxit = c->p.max_iter;
    int rc = PCE_OK;
    const bool use_graph = !c->timing && graphs_enabled() && !c->cg_graph_failed;
    if (use_graph && (!c->cg_graph || c->cg_graph_stale)) {
        if ((rc = capture_iteration(c))) return rc;
    }
    // iterations kept in flight: large meshes take milliseconds per iteration (an unneeded replay costs its cuFFT passes), small
    // ones are launch-bound
    const long long mesh = (long long)c->p.Ng[0] * c->p.Ng[1] * c->p.Ng[2];
    const int depth = (mesh >= (1ll << 24)) ? 1 : 3;
    int launched = 0;
    for (;;) {
        if (launched >= depth && (rc = wait_progress(c, launched - depth + 1))) return rc;
        if (c->cg_host->done || launched >= maxit) break;
        if (use_graph && c->cg_graph) {
            PCE_CUDA(c, cudaGraphLaunch(c->cg_graph, c->st));
            c->launches += c->cg_graph_launches;
            inf->graph_replays++;
        } else if ((rc = enqueue_iteration(c))) return rc;
        ++launched;
    }
    if ((rc = wait_progress(c, launched))) return rc;
    inf->iters = c->cg_host->it;
    inf->matvecs += c->cg_host->it;
    const double gg = c->cg_host->gg, ref = c->cg_host->ref;
    inf->rel_resid = sqrt(gg) / ref;
    if (!(gg == gg)) { c->err = "NaN in the Krylov residual"; return PCE_ECUDA; }
    inf->converged = (inf->rel_resid <= c->p.tol_solver) ? 1 : 0;
    return PCE_OK;
}

int solve_cg(pce_ctx* c, const double* Q_body, const double* q_ion, const double E0[3], int warm, double* q, double* Phi,
             pce_solve_info* info)
{
    const int nb = c->Nbody, nbead = c->Nbead;
    pce_solve_info inf = {0, 0, 0.0, 1};
    int rc = krylov_alloc(c);
    if (rc) return rc;
    // 1. starting charges (beads in the context's own iterate, ions fixed)
    if (nb > 0 && nbead > 0) {
        PassTimer t(c, PASS_KRYLOV);
        k_init_q<<<nb, BT, 0, c->st>>>(c->body_off, Q_body, warm, q, c->cg_q);
        k_copy<<<cdiv(nbead, 256), 256, 0, c->st>>>(nbead, c->cg_q, q);
        c->launches += 2;
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
    if ((rc = op_evaluate_at_beads(c, q, c->cg_psi))) return rc;
    inf.matvecs = 1;
    c->cg_host->it = -1; c->cg_host->done = 0;
    {
        PassTimer t(c, PASS_KRYLOV);
        k_resid_init<<<nb, BT, 0, c->st>>>(nb, c->body_off, c->rx, c->ry, c->rz, E0[0], E0[1], E0[2], c->cg_psi, c->cg_g, c->cg_part, c->cg_state,
                                         c->cg_host_dev, warm, c->pc_on ? 1 : 0, c->p.tol_solver, c->p.max_iter);
        c->launches++;
        if (c->pc_on && (rc = enqueue_precond(c, 1))) return rc;
    }
    PCE_CUDA(c, cudaGetLastError());
    if ((rc = wait_progress(c, 0))) return rc;
    if ((rc = run_iterations(c, &inf))) return rc;
    {
        PassTimer t(c, PASS_KRYLOV);
        k_body_mean<<<nb, BT, 0, c->st>>>(c->body_off, c->cg_psi, c->rx, c->ry, c->rz, E0[0], E0[1], E0[2], Phi);
        k_copy<<<cdiv(nbead, 256), 256, 0, c->st>>>(nbead, c->cg_q, q);
        c->launches += 2;
    }
    PCE_CUDA(c, cudaGetLastError());
    if (info) *info = inf;
    return inf.converged ? PCE_OK : PCE_ENOCONV;
}

// M_bb q = b over the conductor beads, no constraint (a column of the grand capacitance tensor, eq. 15)
int solve_plain(pce_ctx* c, const double* b, double* q, pce_solve_info* info)
{
    const int nbead = c->Nbead;
    pce_solve_info inf = {0, 0, 0.0, 1};
    int rc = krylov_alloc(c);
    if (rc) return rc;
    c->cg_host->it = -1; c->cg_host->done = 0;
    {
        PassTimer t(c, PASS_KRYLOV);
        k_resid_init_plain<<<pupdate_blocks(c), BT, 0, c->st>>>(nbead, b, c->cg_g, c->cg_q, c->cg_psi, c->cg_part, c->cg_state, c->cg_host_dev,
                                                               c->pc_on ? 1 : 0, c->p.tol_solver, c->p.max_iter);
        c->launches++;
        if (c->pc_on && (rc = enqueue_precond(c, 1))) return rc;
    }
    PCE_CUDA(c, cudaGetLastError());
    if ((rc = wait_progress(c, 0))) return rc;
    if ((rc = run_iterations(c, &inf))) return rc;
    k_copy<<<cdiv(nbead, 256), 256, 0, c->st>>>(nbead, c->cg_q, q);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    if (info) *info = inf;
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

// ---------------------------------------------------------------- grand capacitance tensor (eq. 15) and eps_eff (eq. 36)
// right-hand side Sigma'^T e_k: column k < N_body: 1 on the beads of body k; column N_body + 3 i + d: r_ij,d on the beads of body i
__global__ void k_cap_rhs(int n, int nb, int col, const int* __restrict__ body_of, const double* __restrict__ rx, const double* __restrict__ ry,
                          const double* __restrict__ rz, double* __restrict__ b)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const int body = body_of[j];
    double v = 0.0;
    if (col < nb) v = (body == col) ? 1.0 : 0.0;
    else {
        const int i = (col - nb) / 3, d = (col - nb) % 3;
        if (body == i) v = (d == 0) ? rx[j] : (d == 1) ? ry[j] : rz[j];
    }
    b[j] = v;
}

// moments [Q; S] = Sigma' q: out[i] = sum_j q_ij, out[nb + 3 i + d] = sum_j r_ij,d q_ij (one CTA per body, fixed order)
__global__ void __launch_bounds__(BT)
k_cap_moments(int nb, const int* __restrict__ off, const double* __restrict__ q, const double* __restrict__ rx, const double* __restrict__ ry,
              const double* __restrict__ rz, double* __restrict__ out)
{
    __shared__ double sh[32];
    const int b = blockIdx.x;
    const int j0 = off[b], j1 = off[b + 1];
    double a[4] = {0, 0, 0, 0};
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const double qj = q[j];
        a[0] += qj; a[1] += rx[j] * qj; a[2] += ry[j] * qj; a[3] += rz[j] * qj;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) a[k] = block_sum(a[k], sh);
    if (threadIdx.x == 0) { out[b] = a[0]; out[nb + 3 * b] = a[1]; out[nb + 3 * b + 1] = a[2]; out[nb + 3 * b + 2] = a[3]; }
}

int capacitance_columns(pce_ctx* c, int ncol, const int* cols, double* C, pce_solve_info* info)
{
    const int nb = c->Nbody, n = c->Nbead;
    pce_solve_info worst = {0, 0, 0.0, 1};
    int rc_all = PCE_OK;
    for (int k = 0; k < ncol; ++k) {
        const int col = cols[k];
        if (col < 0 || col >= 4 * nb) { c->err = "pce_capacitance_columns: column index out of range"; return PCE_EINVAL; }
        double *b = c->ev_psi, *q = c->ev_ex;  // the evaluation work vectors are free between operator calls
        k_cap_rhs<<<cdiv(n, 256), 256, 0, c->st>>>(n, nb, col, c->body_of, c->rx, c->ry, c->rz, b);
        c->launches++;
        pce_solve_info inf;
        int rc = solve_plain(c, b, q, &inf);
        if (rc != PCE_OK && rc != PCE_ENOCONV) return rc;
        if (rc == PCE_ENOCONV) rc_all = PCE_ENOCONV;
        k_cap_moments<<<nb, BT, 0, c->st>>>(nb, c->body_off, q, c->rx, c->ry, c->rz, C + (size_t)k * 4 * nb);
        c->launches++;
        worst.iters = worst.iters > inf.iters ? worst.iters : inf.iters;
        worst.matvecs += inf.matvecs;
        worst.graph_replays += inf.graph_replays;
        worst.rel_resid = worst.rel_resid > inf.rel_resid ? worst.rel_resid : inf.rel_resid;
        worst.converged = worst.converged && inf.converged;
    }
    PCE_CUDA(c, cudaGetLastError());
    if (info) *info = worst;
    return rc_all;
}

// eq. 36: eps_eff = eps_f - n <C_SPsi C_qPsi^-1 C_qE - C_SE>.  The bracket is the mean dipole response of
// floating bodies (Q = 0: the potentials adjust) to a unit field that is the same on every body, i.e. the constrained solve
// of eq. 13 with E0 = e_d, Q = 0 and no ionic charge: column d of eps_eff - eps_f I is (1/V) sum_i S_i.
int effective_permittivity(pce_ctx* c, double eps_eff[9], pce_solve_info* info)
{
    const int nb = c->Nbody, N = c->N;
    pce_solve_info worst = {0, 0, 0.0, 1};
    int rc_all = PCE_OK;
    // ev_psi holds max(N, 4 N_body) doubles (pce_set_system): room for the 4 N_body moments of k_cap_moments
    double *zeros = c->ev_ey, *q = c->ev_ez, *Phi = c->ev_ex, *mom = c->ev_psi;
    // the three unit-field solves below are cold starts of a problem of their own scale: keep the residual scale of the caller's
    // last cold pce_solve, which its next warm-started solve measures its tolerance against
    int rc0 = krylov_alloc(c);
    if (rc0) return rc0;
    struct RefColdKeeper {
        pce_ctx* c;
        explicit RefColdKeeper(pce_ctx* c_) : c(c_) { k_ref_cold_keep<<<1, 1, 0, c->st>>>(c->cg_state, 0); c->launches++; }
        ~RefColdKeeper() { k_ref_cold_keep<<<1, 1, 0, c->st>>>(c->cg_state, 1); c->launches++; }
    } keep(c);
    PCE_CUDA(c, cudaMemsetAsync(zeros, 0, (size_t)N * sizeof(double), c->st));
    std::vector<double> h((size_t)4 * nb);
    for (int d = 0; d < 3; ++d) {
        const double E0[3] = {d == 0 ? 1.0 : 0.0, d == 1 ? 1.0 : 0.0, d == 2 ? 1.0 : 0.0};
        pce_solve_info inf;
        int rc = solve_cg(c, zeros, zeros, E0, 0, q, Phi, &inf);
        if (rc != PCE_OK && rc != PCE_ENOCONV) return rc;
        if (rc == PCE_ENOCONV) rc_all = PCE_ENOCONV;
        k_cap_moments<<<nb, BT, 0, c->st>>>(nb, c->body_off, q, c->rx, c->ry, c->rz, mom);
        c->launches++;
        PCE_CUDA(c, cudaMemcpyAsync(h.data(), mom, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->st));
        PCE_CUDA(c, cudaStreamSynchronize(c->st));
        for (int e = 0; e < 3; ++e) {
            double s = 0.0;
            for (int i = 0; i < nb; ++i) s += h[(size_t)nb + 3 * i + e];
            eps_eff[3 * e + d] = (e == d ? c->p.eps_f : 0.0) + s / c->V;
        }
        worst.iters = worst.iters > inf.iters ? worst.iters : inf.iters;
        worst.matvecs += inf.matvecs;
        worst.graph_replays += inf.graph_replays;
        worst.rel_resid = worst.rel_resid > inf.rel_resid ? worst.rel_resid : inf.rel_resid;
        worst.converged = worst.converged && inf.converged;
    }
    if (info) *info = worst;
    return rc_all;
}
