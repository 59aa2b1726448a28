// pce_api.cu -- the C ABI of include/pce.h: context, parameter derivation
// (eqs. 23, 28, 31, 32), orchestration of the spectral Ewald passes
// (steps 1-6) and per-pass timing.
#include "pce_internal.h"

#include <cmath>

static std::string g_create_err;

// ---------------------------------------------------------------- parameters
extern "C" int pce_suggest_params(const double L[3], const int Ng[3], double a, double tol, int P_override, pce_params* out)
{
    if (!L || !Ng || !out || !(tol > 0.0 && tol < 1.0) || !(a > 0.0)) return PCE_EINVAL;
    for (int d = 0; d < 3; ++d)
        if (!(L[d] > 0.0) || Ng[d] < 4) return PCE_EINVAL;
    const double s = std::sqrt(-std::log(tol));
    double kc = 1e300;
    for (int d = 0; d < 3; ++d) kc = std::fmin(kc, PCE_PI * (Ng[d] - 1) / L[d]);  // N_g = 1 + L k_c / pi
    const double xi = kc / (2.0 * s);                                            // exp(-k_c^2/4xi^2) = tol (eq. 28)
    const double rc = s / xi + 2.0 * a;                                          // eq. 23, shells: erfc((r-2a) xi)
    int P = P_override;
    if (P <= 0) {
        const double p0 = (2.0 / PCE_PI) * (-std::log(tol)) + 4.0;               // exp(-pi P/2) <~ tol e^{-2 pi} (eq. 32)
        P = 2 * (int)std::ceil(p0 / 2.0);
    }
    if (P < 4) P = 4;
    if (P > 32) P = 32;
    for (int d = 0; d < 3; ++d)
        if (P > Ng[d]) P = Ng[d] & ~1;
    std::memset(out, 0, sizeof(*out));
    for (int d = 0; d < 3; ++d) { out->L[d] = L[d]; out->Ng[d] = Ng[d]; }
    out->xi = xi; out->rc = rc; out->P = P; out->a = a; out->eps_f = 1.0;
    out->P_matvec = P;  // the same window for the solver matvec (a narrower one is the caller's choice, pce.h)
    out->tol_solver = 1e-12; out->max_iter = 500; out->flags = 0;
    return PCE_OK;
}

// ---------------------------------------------------------------- timing
void timing_begin(pce_ctx* c)
{
    std::memset(&c->tm, 0, sizeof(c->tm));
    c->recs.clear();
    c->ev_used = 0;
}

void timing_end(pce_ctx* c)
{
    if (!c->timing) return;
    cudaStreamSynchronize(c->st);
    double* slot[PASS_COUNT] = {&c->tm.cells, &c->tm.real, &c->tm.spread, &c->tm.fft, &c->tm.scale,
                                &c->tm.ifft,  &c->tm.gather, &c->tm.krylov, &c->tm.other};
    for (auto& r : c->recs) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, r.a, r.b);
        *slot[r.pass] += ms;
        c->tm.total += ms;
        if (r.bead) {
            if (r.pass == PASS_REAL) c->tm.bead_real += ms;
            if (r.pass == PASS_SPREAD) c->tm.bead_spread += ms;
            if (r.pass == PASS_GATHER) c->tm.bead_gather += ms;
        }
    }
    c->recs.clear();
    c->ev_used = 0;
}

// ---------------------------------------------------------------- create / destroy
static void free_system(pce_ctx* c)
{
    cudaFree(c->x); cudaFree(c->y); cudaFree(c->z); cudaFree(c->body_off); cudaFree(c->body_of);
    cudaFree(c->rx); cudaFree(c->ry); cudaFree(c->rz); cudaFree(c->X); cudaFree(c->Y); cudaFree(c->Z);
    bins_free(c->all); bins_free(c->bead); bins_free(c->wall); bins_free(c->wbead); bins_free(c->wbead_s);
    cudaFree(c->csr_ptr); cudaFree(c->csr_col); cudaFree(c->csr_val);
    cudaFree(c->w_real); cudaFree(c->w_wave); cudaFree(c->w_ex); cudaFree(c->w_ey); cudaFree(c->w_ez);
    cudaFree(c->w_kx); cudaFree(c->w_ky); cudaFree(c->w_kz);
    cudaFree(c->cg_g); cudaFree(c->cg_p); cudaFree(c->cg_t); cudaFree(c->cg_ap); cudaFree(c->cg_psi); cudaFree(c->cg_q);
    cudaFree(c->ev_psi); cudaFree(c->ev_ex); cudaFree(c->ev_ey); cudaFree(c->ev_ez); cudaFree(c->cg_part);
    krylov_invalidate_graph(c);
    cudaFree(c->hs_dev); cudaFree(c->cg_z); cudaFree(c->pc_mean);
    precond_free(c);
    dynamics_free(c);
    c->cg_z = c->pc_mean = nullptr;
    c->x = c->y = c->z = nullptr; c->body_off = c->body_of = nullptr;
    c->rx = c->ry = c->rz = c->X = c->Y = c->Z = nullptr;
    c->csr_ptr = c->csr_col = nullptr; c->csr_val = nullptr; c->nnz = c->nnz_cap = 0;
    c->w_real = c->w_wave = c->w_ex = c->w_ey = c->w_ez = c->w_kx = c->w_ky = c->w_kz = nullptr;
    c->cg_g = c->cg_p = c->cg_t = c->cg_ap = c->cg_psi = c->cg_q = nullptr;
    c->ev_psi = c->ev_ex = c->ev_ey = c->ev_ez = c->cg_part = nullptr;
    c->hs_dev = nullptr; c->hs_dev_n = 0;
    c->have_system = false;
    if (c->cg_state) cudaMemsetAsync(c->cg_state, 0, sizeof(CgState), c->st);  // forget the residual scale of the old system
    c->bytes = c->bytes_base;
}

extern "C" int pce_destroy(pce_ctx* c)
{
    if (!c) return PCE_EINVAL;
    cudaStreamSynchronize(c->st);
    free_system(c);
    krylov_free(c);
    if (c->have_plans) { cufftDestroy(c->planF); cufftDestroy(c->planB); }
    cudaFree(c->fft_work); cudaFree(c->grid); cudaFree(c->gridk); cudaFree(c->gridk2); cudaFree(c->scal); cudaFree(c->sum_part); cudaFree(c->scan_tmp); cudaFree(c->work_ctr); cudaFree(c->rt_dev); cudaFree(c->ztw); cudaFree(c->zexp_set[0]); cudaFree(c->zexp_set[1]); cudaFree(c->zshape); cudaFree(c->xytw); cudaFree(c->xy_ctr); cudaFree(c->gather_part);
    for (auto e : c->ev_pool) cudaEventDestroy(e);
    delete c;
    return PCE_OK;
}

extern "C" const char* pce_last_error(const pce_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

// wave-space constants of a window with P support points per dimension (eq. 25, 31: eta = h^2 xi^2 P / pi)
static void wave_const_for(const pce_ctx* c, int P, WaveConst& w)
{
    const pce_params& p = c->p;
    double cn2 = 1.0, h3 = 1.0, ntot = 1.0;
    for (int d = 0; d < 3; ++d) {
        const double h = p.L[d] / p.Ng[d], eta = h * h * p.xi * p.xi * P / PCE_PI;
        w.Ng[d] = p.Ng[d]; w.L[d] = p.L[d]; w.h[d] = h; w.inv_h[d] = 1.0 / h;
        w.kfac[d] = 2.0 * PCE_PI / p.L[d];
        w.gexp[d] = (1.0 - eta) / (4.0 * p.xi * p.xi);
        w.grad_fac[d] = 4.0 * PCE_PI / (P * h);
        cn2 *= 2.0 / (P * h * h);
        h3 *= h;
        ntot *= p.Ng[d];
    }
    w.Nxh = p.Ng[0] / 2 + 1;
    w.P = P;
    w.aw = 2.0 * PCE_PI / P;
    w.a = p.a;
    w.scale_norm = cn2 * h3 / (p.eps_f * ntot);
    for (int r = 0; r < 32; ++r) w.G[r] = std::exp(-w.aw * r * r);
}

// the window of the next wave passes: 0 = P (evaluations with fields, right-hand side), 1 = P_matvec (solver matvec)
void wave_select(pce_ctx* c, int which)
{
    c->wk = c->wset[which];
    c->zexp = c->zexp_set[which];
}

static int create_impl(pce_ctx* c)
{
    const pce_params& p = c->p;
    c->V = p.L[0] * p.L[1] * p.L[2];
    for (int d = 0; d < 3; ++d) {
        c->h[d] = p.L[d] / p.Ng[d];
        c->eta[d] = c->h[d] * c->h[d] * p.xi * p.xi * p.P / PCE_PI;  // eq. 31
    }
    c->P_mv = (p.P_matvec >= 4 && p.P_matvec < p.P) ? p.P_matvec : p.P;
    wave_const_for(c, p.P, c->wset[0]);
    wave_const_for(c, c->P_mv, c->wset[1]);
    c->wk = c->wset[0];
    WaveConst& w = c->wk;
    RealConst& r = c->rk;
    r.a = p.a; r.xi = p.xi; r.two_a = 2.0 * p.a; r.inv_eps = 1.0 / p.eps_f;
    r.c64 = 1.0 / (64.0 * PCE_PI * p.a * p.a * p.xi * p.xi);
    r.rc2 = p.rc * p.rc;
    const double pi32 = PCE_PI * std::sqrt(PCE_PI);
    const double e4 = std::exp(-4.0 * p.a * p.a * p.xi * p.xi);
    r.R0 = (1.0 - e4) / (8.0 * pi32 * p.a * p.a * p.xi) + std::erfc(2.0 * p.a * p.xi) / (4.0 * PCE_PI * p.a);  // eq. 21
    r.two_xi_sqrtpi = 2.0 * p.xi / std::sqrt(PCE_PI);
    r.t_lin = 1.0 / (16.0 * PCE_PI * p.a * p.a);
    r.t_quad = p.xi * (1.0 - e4) / (24.0 * pi32 * p.a * p.a);
    r.r_small = 1e-3 * p.a;
    c->kconst = 1.0 / (4.0 * p.xi * p.xi * c->V * p.eps_f);  // k = 0 removal (reading A1)

    const size_t ng = (size_t)p.Ng[0] * p.Ng[1] * p.Ng[2];
    const size_t nk = (size_t)w.Nxh * p.Ng[1] * p.Ng[2];
    if (cudaMalloc(&c->grid, ng * sizeof(double)) != cudaSuccess || cudaMalloc(&c->gridk, nk * sizeof(cufftDoubleComplex)) != cudaSuccess) {
        c->err = "out of device memory for the FFT grids";
        return PCE_ENOMEM;
    }
    c->bytes += (long long)(ng * 8 + nk * 16);
    PCE_CUDA(c, cudaMalloc(&c->scal, 64 * sizeof(double)));
    PCE_CUDA(c, cudaMalloc(&c->sum_part, 1024 * sizeof(double)));
    // cuFFT plans sharing one work area
    size_t wsF = 0, wsB = 0;
    if (cufftCreate(&c->planF) != CUFFT_SUCCESS || cufftCreate(&c->planB) != CUFFT_SUCCESS) { c->err = "cufftCreate failed"; return PCE_ECUFFT; }
    c->have_plans = true;
    cufftSetAutoAllocation(c->planF, 0);
    cufftSetAutoAllocation(c->planB, 0);
    c->use_zfft = zfft_supported(p) && !(p.flags & PCE_FLAG_CUFFT_3D);
    if (c->use_zfft) {  // (x, y) transforms per mesh plane by cuFFT, the z axis fused with the scaling (zfft.cu)
        int dims[2] = {p.Ng[1], p.Ng[0]};
        if (cufftMakePlanMany(c->planF, 2, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, p.Ng[2], &wsF) != CUFFT_SUCCESS ||
            cufftMakePlanMany(c->planB, 2, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_Z2D, p.Ng[2], &wsB) != CUFFT_SUCCESS) {
            c->err = "cuFFT cannot plan this grid";
            return PCE_ECUFFT;
        }
        int rcz = zfft_init(c);
        if (rcz) return rcz;
        c->use_fftxy = fftxy_supported(p);
        if (c->use_fftxy && (rcz = fftxy_init(c))) return rcz;
    } else if (cufftMakePlan3d(c->planF, p.Ng[2], p.Ng[1], p.Ng[0], CUFFT_D2Z, &wsF) != CUFFT_SUCCESS ||
               cufftMakePlan3d(c->planB, p.Ng[2], p.Ng[1], p.Ng[0], CUFFT_Z2D, &wsB) != CUFFT_SUCCESS) {
        c->err = "cuFFT cannot plan this grid";
        return PCE_ECUFFT;
    }
    const size_t ws = wsF > wsB ? wsF : wsB;
    if (ws > 0) {
        if (cudaMalloc(&c->fft_work, ws) != cudaSuccess) { c->err = "out of device memory for the cuFFT work area"; return PCE_ENOMEM; }
        c->bytes += (long long)ws;
    }
    cufftSetWorkArea(c->planF, c->fft_work);
    cufftSetWorkArea(c->planB, c->fft_work);
    cufftSetStream(c->planF, c->st);
    cufftSetStream(c->planB, c->st);
    int rcw = wave_bricks_init(c);
    if (rcw) return rcw;
    c->use_cols = wave_cols_supported(c);
    if ((p.flags & PCE_FLAG_DETERMINISTIC) && !c->use_cols) {
        c->err = "PCE_FLAG_DETERMINISTIC needs a mesh on the brick lattice (N_g % 8 == 0, N_g - P >= 8)";
        return PCE_EINVAL;
    }
    if (c->use_cols && (rcw = wave_cols_init(c))) return rcw;
    return realtab_upload(c);
}

extern "C" int pce_create(const pce_params* p, void* stream, pce_ctx** out)
{
    if (!p || !out) { g_create_err = "NULL argument"; return PCE_EINVAL; }
    *out = nullptr;
    bool ok = p->xi > 0 && p->rc > 0 && p->a > 0 && p->eps_f > 0 && p->P >= 4 && p->P <= 32 && (p->P % 2 == 0) && p->max_iter > 0 &&
              p->tol_solver > 0;
    for (int d = 0; d < 3 && ok; ++d) ok = p->L[d] > 0 && p->Ng[d] >= p->P && p->Ng[d] >= 4;
    if (ok && p->P_matvec != 0) ok = p->P_matvec >= 4 && p->P_matvec <= p->P && p->P_matvec % 2 == 0;
    if (!ok) { g_create_err = "invalid pce_params (need xi,rc,a,eps_f>0; P even in 4..32; P_matvec 0 or even in 4..P; Ng>=P; max_iter>0)"; return PCE_EINVAL; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        g_create_err = "no CUDA device: this library has no CPU fallback";
        return PCE_ECUDA;
    }
    pce_ctx* c = new pce_ctx();
    c->p = *p;
    c->st = (cudaStream_t)stream;
    std::memset(&c->tm, 0, sizeof(c->tm));
    int rc = create_impl(c);
    c->bytes_base = c->bytes;
    if (rc != PCE_OK) {
        g_create_err = c->err;
        pce_destroy(c);
        return rc;
    }
    *out = c;
    return PCE_OK;
}

// ---------------------------------------------------------------- system / positions
static void cell_layout(const pce_params& p, int nc[3], int range[3])
{
    for (int d = 0; d < 3; ++d) {
        int n = (int)std::floor(p.L[d] / p.rc);
        if (n > 256) n = 256;
        if (n >= 3) { nc[d] = n; range[d] = 1; }
        else { nc[d] = 1; range[d] = (int)std::ceil(p.rc / p.L[d]); }  // explicit periodic images (reading A10)
    }
}

#define ALLOC_D(ptr, n)                                                                                     \
    do {                                                                                                    \
        size_t n__ = (size_t)((n) > 0 ? (n) : 1);                                                           \
        if (cudaMalloc(&(ptr), n__ * sizeof(double)) != cudaSuccess) { c->err = "out of device memory"; return PCE_ENOMEM; } \
        c->bytes += (long long)(n__ * 8);                                                                   \
    } while (0)

static int positions_impl(pce_ctx* c, const double* x, const double* y, const double* z)
{
    int rc;
    krylov_invalidate_graph(c);  // list sizes, grid dimensions and possibly reallocated buffers are baked into the captured iteration
    {
        PassTimer t(c, PASS_CELLS);
        if ((rc = wrap_positions(c, c->N, x, y, z, c->x, c->y, c->z))) return rc;
        if ((rc = bins_build(c, c->all, c->x, c->y, c->z))) return rc;
        if ((rc = bins_build(c, c->bead, c->x, c->y, c->z))) return rc;  // beads are the first Nbead particles
        if ((rc = bins_build(c, c->wall, c->x, c->y, c->z))) return rc;
        if ((rc = bins_build(c, c->wbead, c->x, c->y, c->z))) return rc;
        if (c->use_cols) {
            if ((rc = wave_cols_build(c, c->wall))) return rc;
            if ((rc = wave_cols_build(c, c->wbead))) return rc;
        } else {
            if ((rc = wave_window_coef(c, c->wall))) return rc;
            if ((rc = wave_window_coef(c, c->wbead))) return rc;
        }
        if (c->wmv == &c->wbead_s) {  // the beads once more for the narrower window of the solver matvec
            wave_select(c, 1);
            rc = bins_build(c, c->wbead_s, c->x, c->y, c->z);
            if (!rc) rc = c->use_cols ? wave_cols_build(c, c->wbead_s) : wave_window_coef(c, c->wbead_s);
            wave_select(c, 0);
            if (rc) return rc;
        }
        if ((rc = bodies_setup(c))) return rc;
    }
    if ((rc = real_csr_build(c, c->bead))) return rc;
    return PCE_OK;
}

int positions_update(pce_ctx* c, const double* x, const double* y, const double* z) { return positions_impl(c, x, y, z); }

extern "C" int pce_set_system(pce_ctx* c, int N, int N_body, const int* body_offset, const double* x, const double* y, const double* z)
{
    if (!c) return PCE_EINVAL;
    if (N <= 0 || N_body < 0 || !x || !y || !z || (N_body > 0 && !body_offset)) { c->err = "pce_set_system: bad arguments"; return PCE_EINVAL; }
    std::vector<int> off(N_body + 1, 0);
    for (int i = 0; i <= N_body && N_body > 0; ++i) off[i] = body_offset[i];
    if (off[0] != 0) { c->err = "body_offset[0] must be 0"; return PCE_EINVAL; }
    for (int i = 0; i < N_body; ++i)
        if (off[i + 1] < off[i]) { c->err = "body_offset must be non-decreasing"; return PCE_EINVAL; }
    if (off[N_body] > N) { c->err = "body_offset[N_body] exceeds N"; return PCE_EINVAL; }
    timing_begin(c);
    cudaStreamSynchronize(c->st);
    free_system(c);
    c->N = N; c->Nbody = N_body; c->Nbead = off[N_body]; c->Nion = N - c->Nbead;
    c->body_off_h = off;
    const int nb1 = N_body + 1;
    ALLOC_D(c->x, N); ALLOC_D(c->y, N); ALLOC_D(c->z, N);
    ALLOC_D(c->rx, c->Nbead); ALLOC_D(c->ry, c->Nbead); ALLOC_D(c->rz, c->Nbead);
    ALLOC_D(c->X, N_body); ALLOC_D(c->Y, N_body); ALLOC_D(c->Z, N_body);
    PCE_CUDA(c, cudaMalloc(&c->body_off, (size_t)nb1 * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&c->body_of, (size_t)(c->Nbead > 0 ? c->Nbead : 1) * sizeof(int)));
    PCE_CUDA(c, cudaMemcpyAsync(c->body_off, off.data(), (size_t)nb1 * sizeof(int), cudaMemcpyHostToDevice, c->st));
    {
        std::vector<int> bo((size_t)(c->Nbead > 0 ? c->Nbead : 1), 0);
        for (int b = 0; b < N_body; ++b)
            for (int j = off[b]; j < off[b + 1]; ++j) bo[j] = b;
        PCE_CUDA(c, cudaMemcpyAsync(c->body_of, bo.data(), bo.size() * sizeof(int), cudaMemcpyHostToDevice, c->st));
        PCE_CUDA(c, cudaStreamSynchronize(c->st));
    }
    int nc[3], range[3], rc;
    cell_layout(c->p, nc, range);
    if ((rc = bins_alloc(c, c->all, N, nc, range))) return rc;
    if ((rc = bins_alloc(c, c->bead, c->Nbead, nc, range))) return rc;
    if ((rc = bins_alloc_chunks(c, c->all))) return rc;
    if ((rc = bins_alloc_chunks(c, c->bead))) return rc;
    if ((rc = bins_alloc_tiles(c, c->wall, N, 8))) return rc;  // 8-point mesh bins = bricks of wave_bricks.cu
    if ((rc = bins_alloc_tiles(c, c->wbead, c->Nbead, 8))) return rc;
    if (c->use_cols) {
        if ((rc = wave_cols_alloc(c, c->wall))) return rc;
        if ((rc = wave_cols_alloc(c, c->wbead))) return rc;
    } else {
        if ((rc = wave_coef_alloc(c, c->wall))) return rc;
        if ((rc = wave_coef_alloc(c, c->wbead))) return rc;
    }
    c->wmv = &c->wbead;
    if (c->P_mv != c->p.P && c->Nbead > 0) {
        wave_select(c, 1);
        rc = bins_alloc_tiles(c, c->wbead_s, c->Nbead, 8);
        if (!rc) rc = c->use_cols ? wave_cols_alloc(c, c->wbead_s) : wave_coef_alloc(c, c->wbead_s);
        wave_select(c, 0);
        if (rc) return rc;
        c->wmv = &c->wbead_s;
    }
    PCE_CUDA(c, cudaMalloc(&c->csr_ptr, ((size_t)c->Nbead + 2) * sizeof(int)));
    ALLOC_D(c->w_real, N); ALLOC_D(c->w_wave, N); ALLOC_D(c->w_ex, N); ALLOC_D(c->w_ey, N); ALLOC_D(c->w_ez, N);
    ALLOC_D(c->w_kx, N); ALLOC_D(c->w_ky, N); ALLOC_D(c->w_kz, N);
    ALLOC_D(c->cg_g, c->Nbead); ALLOC_D(c->cg_p, c->Nbead); ALLOC_D(c->cg_t, c->Nbead); ALLOC_D(c->cg_ap, c->Nbead);
    ALLOC_D(c->cg_psi, c->Nbead); ALLOC_D(c->cg_q, c->Nbead);
    ALLOC_D(c->ev_psi, N > 4 * N_body ? N : 4 * N_body);  // also the 4 N_body body moments of pce_effective_permittivity
    ALLOC_D(c->ev_ex, N); ALLOC_D(c->ev_ey, N); ALLOC_D(c->ev_ez, N);
    ALLOC_D(c->cg_part, 3 * (N_body > 1024 ? N_body : 1024));
    ALLOC_D(c->cg_z, c->Nbead); ALLOC_D(c->pc_mean, N_body);
    c->have_system = true;
    rc = positions_impl(c, x, y, z);
    if (!rc) rc = precond_setup(c);  // needs r_ij of bodies_setup; rigid bodies: once per system
    timing_end(c);
    return rc;
}

extern "C" int pce_set_positions(pce_ctx* c, const double* x, const double* y, const double* z)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_set_positions before pce_set_system"; return PCE_ESTATE; }
    if (!x || !y || !z) { c->err = "NULL positions"; return PCE_EINVAL; }
    timing_begin(c);
    int rc = positions_impl(c, x, y, z);
    timing_end(c);
    return rc;
}

extern "C" int pce_set_centres(pce_ctx* c, const double* X, const double* Y, const double* Z)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_set_centres before pce_set_system"; return PCE_ESTATE; }
    if (c->Nbody > 0 && (!X || !Y || !Z)) { c->err = "NULL centres"; return PCE_EINVAL; }
    return bodies_set_centres(c, X, Y, Z);
}

// ---------------------------------------------------------------- the operator
// out[0] = sum(in[0..n)): per-block partials, then one block (fixed order: deterministic)
__global__ void __launch_bounds__(256) k_sum_partial(const double* __restrict__ in, int n, double* __restrict__ part)
{
    __shared__ double sh[8];
    double v = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) v += in[i];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < 8; ++i) s += sh[i];
        part[blockIdx.x] = s;
    }
}

__global__ void __launch_bounds__(256) k_sum_final(const double* __restrict__ part, int nb, double* __restrict__ out)
{
    __shared__ double sh[8];
    double v = 0.0;
    for (int i = threadIdx.x; i < nb; i += blockDim.x) v += part[i];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < 8; ++i) s += sh[i];
        out[0] = s;
    }
}

int sum_vector(pce_ctx* c, const double* in, int n, double* out)
{
    int nb = cdiv(n, 256 * 8);
    if (nb > 1024) nb = 1024;
    if (nb < 1) nb = 1;
    k_sum_partial<<<nb, 256, 0, c->st>>>(in, n, c->sum_part);
    k_sum_final<<<1, 256, 0, c->st>>>(c->sum_part, nb, out);
    c->launches += 2;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// caller order j: psi[j] = real[inv_r[j]] + wave[inv_w[j]] - (sum q)/(4 xi^2 V eps); fields likewise (no constant)
__global__ void k_finalize(int n, const int* __restrict__ inv_r, const int* __restrict__ inv_w, const double* __restrict__ re,
                           const double* __restrict__ wa, const double* __restrict__ qsum, double kconst, double* __restrict__ psi,
                           int field, const double* __restrict__ rx, const double* __restrict__ ry, const double* __restrict__ rz,
                           const double* __restrict__ kx, const double* __restrict__ ky, const double* __restrict__ kz,
                           double* __restrict__ ex, double* __restrict__ ey, double* __restrict__ ez)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const int ir = inv_r[j], iw = inv_w[j];
    psi[j] = re[ir] + wa[iw] - kconst * qsum[0];
    if (field) { ex[j] = rx[ir] + kx[iw]; ey[j] = ry[ir] + ky[iw]; ez[j] = rz[ir] + kz[iw]; }
}

// sources: the particle subset (sr: real-space cells, sw: mesh bins) whose charges q (caller order of that subset) act;
// targets: the subset (tr, tw) where potentials / fields are wanted.  Both subsets are prefixes of the particle list.
static int apply_operator(pce_ctx* c, Bins& sr, Bins& sw, Bins& tr, Bins& tw, bool use_csr, const double* q, double* psi, double* Ex,
                          double* Ey, double* Ez)
{
    const bool field = (Ex != nullptr);
    const int n = tr.n;
    int rc;
    {
        PassTimer t(c, PASS_OTHER);
        if ((rc = gather_by_perm(c, sr.n, sr.perm, q, sr.qs))) return rc;
        if ((rc = gather_by_perm(c, sw.n, sw.perm, q, c->use_cols ? sw.qs_cols : sw.qs, c->use_cols ? HITREC_Q_STRIDE : 1))) return rc;
        if ((rc = sum_vector(c, q, sr.n, c->scal))) return rc;
    }
    if (use_csr) rc = real_csr_spmv(c, sr, c->w_real);                                      // step 1 (cached), eq. 20-21
    else rc = real_direct(c, tr, sr, field, c->w_real, c->w_ex, c->w_ey, c->w_ez);          // step 1, eq. 20-21
    if (rc) return rc;
    if ((rc = c->use_cols ? wave_spread_cols(c, sw) : wave_spread_bricks(c, sw))) return rc;  // step 2, eq. 25
    if (field && (c->p.flags & PCE_FLAG_FIELD_IK)) {
        // ik differentiation ("potential and its gradients"): E_d = IFFT[-i k_d G H^] gathered with the plain
        // window -- three more inverse transforms and gathers, but the wave-space forces then sum to zero to rounding
        if ((rc = wave_forward(c))) return rc;                                           // step 3
        double* dst[4] = {c->w_kx, c->w_ky, c->w_kz, c->w_wave};
        for (int k = 0; k < 4; ++k) {
            if ((rc = wave_scale_inverse(c, k < 3 ? k : -1))) return rc;                 // steps 4-5, eq. 26 (times -i k_d)
            if ((rc = c->use_cols ? wave_gather_cols(c, tw, false, dst[k], nullptr, nullptr, nullptr)
                                  : wave_gather_bricks(c, tw, false, dst[k], nullptr, nullptr, nullptr))) return rc;  // step 6
            if (k < 3) c->tm.n_fft_pairs++;
        }
    } else {
        if ((rc = wave_fft_scale_ifft(c))) return rc;                                    // steps 3-5, eq. 26
        if ((rc = c->use_cols ? wave_gather_cols(c, tw, field, c->w_wave, c->w_kx, c->w_ky, c->w_kz)
                              : wave_gather_bricks(c, tw, field, c->w_wave, c->w_kx, c->w_ky, c->w_kz))) return rc;  // step 6, eq. 27
    }
    {
        PassTimer t(c, PASS_OTHER);
        k_finalize<<<cdiv(n, 256), 256, 0, c->st>>>(n, tr.inv, tw.inv, c->w_real, c->w_wave, c->scal, c->kconst, psi, field ? 1 : 0,
                                                   c->w_ex, c->w_ey, c->w_ez, c->w_kx, c->w_ky, c->w_kz, Ex, Ey, Ez);
        c->launches++;
    }
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// the solver's operator (krylov.cu): charges already in the two sorted orders (bead.qs, wbead.qs); results stay sorted
// (w_real, w_wave) and are assembled by the solver's projection kernel
int op_matvec_bead_sorted(pce_ctx* c)
{
    c->tm.n_matvec_bead++;
    c->tm.n_fft_pairs++;
    c->in_bead_matvec = true;
    wave_select(c, 1);  // the solver's window (P_matvec points)
    Bins& wb = *c->wmv;
    int rc = real_csr_spmv(c, c->bead, c->w_real);
    if (!rc) rc = c->use_cols ? wave_spread_cols(c, wb) : wave_spread_bricks(c, wb);
    if (!rc) rc = wave_fft_scale_ifft(c);
    if (!rc) rc = c->use_cols ? wave_gather_cols(c, wb, false, c->w_wave, nullptr, nullptr, nullptr)
                              : wave_gather_bricks(c, wb, false, c->w_wave, nullptr, nullptr, nullptr);
    wave_select(c, 0);
    c->in_bead_matvec = false;
    return rc;
}

int op_matvec_bead(pce_ctx* c, const double* q, double* psi)
{
    c->tm.n_matvec_bead++;
    c->tm.n_fft_pairs++;
    c->in_bead_matvec = true;
    wave_select(c, 1);
    int rc = apply_operator(c, c->bead, *c->wmv, c->bead, *c->wmv, true, q, psi, nullptr, nullptr, nullptr);
    wave_select(c, 0);
    c->in_bead_matvec = false;
    return rc;
}

int op_evaluate(pce_ctx* c, const double* q, double* psi, double* Ex, double* Ey, double* Ez)
{
    c->tm.n_eval_full++;
    c->tm.n_fft_pairs++;
    return apply_operator(c, c->all, c->wall, c->all, c->wall, false, q, psi, Ex, Ey, Ez);
}

// potentials at the conductor beads only, from all N charges (right-hand side of eq. 13): psi has N_bead entries
int op_evaluate_at_beads(pce_ctx* c, const double* q, double* psi)
{
    c->tm.n_eval_full++;
    c->tm.n_fft_pairs++;
    return apply_operator(c, c->all, c->wall, c->bead, c->wbead, false, q, psi, nullptr, nullptr, nullptr);
}

extern "C" int pce_matvec(pce_ctx* c, const double* q, double* psi)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_matvec before pce_set_system"; return PCE_ESTATE; }
    if (!q || !psi) { c->err = "NULL argument"; return PCE_EINVAL; }
    if (c->Nbead == 0) return PCE_OK;
    timing_begin(c);
    int rc = op_matvec_bead(c, q, psi);
    timing_end(c);
    return rc;
}

extern "C" int pce_evaluate(pce_ctx* c, const double* q, double* psi, double* Ex, double* Ey, double* Ez)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_evaluate before pce_set_system"; return PCE_ESTATE; }
    const int nf = (Ex != nullptr) + (Ey != nullptr) + (Ez != nullptr);
    if (!q || !psi || (nf != 0 && nf != 3)) { c->err = "NULL argument (field pointers: all or none)"; return PCE_EINVAL; }
    timing_begin(c);
    int rc = op_evaluate(c, q, psi, Ex, Ey, Ez);
    timing_end(c);
    return rc;
}

extern "C" int pce_solve(pce_ctx* c, const double* Q_body, const double* q_ion, const double E0[3], int warm_start, double* q,
                         double* Phi_body, pce_solve_info* info)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_solve before pce_set_system"; return PCE_ESTATE; }
    if (!E0 || !q || (c->Nbody > 0 && (!Q_body || !Phi_body))) { c->err = "NULL argument"; return PCE_EINVAL; }
    timing_begin(c);
    int rc = solve_cg(c, Q_body, q_ion, E0, warm_start, q, Phi_body, info);
    timing_end(c);
    return rc;
}

extern "C" int pce_forces(pce_ctx* c, const double* q, const double E0[3], double* fx, double* fy, double* fz, double* F, double* T,
                          double* S, double* U_body, double* U_tot, double* psi)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_forces before pce_set_system"; return PCE_ESTATE; }
    if (!q || !E0) { c->err = "NULL argument"; return PCE_EINVAL; }
    timing_begin(c);
    int rc = forces_all(c, q, E0, fx, fy, fz, F, T, S, U_body, U_tot, psi);
    timing_end(c);
    return rc;
}

extern "C" int pce_capacitance_columns(pce_ctx* c, int ncol, const int* cols, double* C, pce_solve_info* info)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_capacitance_columns before pce_set_system"; return PCE_ESTATE; }
    if (ncol < 0 || (ncol > 0 && (!cols || !C))) { c->err = "NULL argument"; return PCE_EINVAL; }
    if (c->Nbody == 0 || c->Nbead == 0) { c->err = "pce_capacitance_columns: the system has no conductor bodies"; return PCE_EINVAL; }
    timing_begin(c);
    int rc = capacitance_columns(c, ncol, cols, C, info);
    timing_end(c);
    return rc;
}

extern "C" int pce_effective_permittivity(pce_ctx* c, double eps_eff[9], pce_solve_info* info)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_effective_permittivity before pce_set_system"; return PCE_ESTATE; }
    if (!eps_eff) { c->err = "NULL argument"; return PCE_EINVAL; }
    if (c->Nbody == 0 || c->Nbead == 0) { c->err = "pce_effective_permittivity: the system has no conductor bodies"; return PCE_EINVAL; }
    timing_begin(c);
    int rc = effective_permittivity(c, eps_eff, info);
    timing_end(c);
    return rc;
}

// ---------------------------------------------------------------- host-buffer pass (bench "e2e")
extern "C" int pce_step_host(pce_ctx* c, const double* x, const double* y, const double* z, const double* Q_body, const double* q_ion,
                             const double E0[3], int warm_start, double* q, double* Phi_body, double* fx, double* fy, double* fz, double* F,
                             double* T, double* S, double* U_tot, pce_solve_info* info)
{
    if (!c) return PCE_EINVAL;
    if (!c->have_system) { c->err = "pce_step_host before pce_set_system"; return PCE_ESTATE; }
    if (!x || !y || !z || !E0 || (c->Nbody > 0 && !Q_body) || (c->Nion > 0 && !q_ion)) { c->err = "NULL argument"; return PCE_EINVAL; }
    if (warm_start && !q) { c->err = "pce_step_host: warm start needs q"; return PCE_EINVAL; }
    const size_t N = c->N, nb = c->Nbody, ni = c->Nion;
    const size_t need = 3 * N + nb + ni + N + nb + 3 * N + 9 * nb + 3 + 8;
    if (need > c->hs_dev_n) {
        cudaFree(c->hs_dev);
        c->hs_dev = nullptr;
        if (cudaMalloc(&c->hs_dev, need * sizeof(double)) != cudaSuccess) { c->err = "out of device memory (host staging)"; c->hs_dev_n = 0; return PCE_ENOMEM; }
        c->hs_dev_n = need;
    }
    double* d = c->hs_dev;
    double *dx = d, *dy = d + N, *dz = d + 2 * N, *dQ = d + 3 * N, *dqi = dQ + nb, *dq = dqi + ni, *dPhi = dq + N;
    double *dfx = dPhi + nb, *dfy = dfx + N, *dfz = dfy + N, *dF = dfz + N, *dT = dF + 3 * nb, *dS = dT + 3 * nb, *dU = dS + 3 * nb;
    timing_begin(c);
    const bool tsave = c->timing;
    PCE_CUDA(c, cudaMemcpyAsync(dx, x, N * 8, cudaMemcpyHostToDevice, c->st));
    PCE_CUDA(c, cudaMemcpyAsync(dy, y, N * 8, cudaMemcpyHostToDevice, c->st));
    PCE_CUDA(c, cudaMemcpyAsync(dz, z, N * 8, cudaMemcpyHostToDevice, c->st));
    if (nb) PCE_CUDA(c, cudaMemcpyAsync(dQ, Q_body, nb * 8, cudaMemcpyHostToDevice, c->st));
    if (ni) PCE_CUDA(c, cudaMemcpyAsync(dqi, q_ion, ni * 8, cudaMemcpyHostToDevice, c->st));
    if (warm_start && c->Nbead) PCE_CUDA(c, cudaMemcpyAsync(dq, q, (size_t)c->Nbead * 8, cudaMemcpyHostToDevice, c->st));
    int rc = positions_impl(c, dx, dy, dz);
    int rc_solve = PCE_OK;
    if (!rc) {
        rc_solve = solve_cg(c, dQ, dqi, E0, warm_start ? 1 : 0, dq, dPhi, info);
        if (rc_solve != PCE_OK && rc_solve != PCE_ENOCONV) rc = rc_solve;
    }
    if (!rc) rc = forces_all(c, dq, E0, dfx, dfy, dfz, dF, dT, dS, nullptr, dU, nullptr);
    if (!rc) {
        if (q) PCE_CUDA(c, cudaMemcpyAsync(q, dq, N * 8, cudaMemcpyDeviceToHost, c->st));
        if (Phi_body && nb) PCE_CUDA(c, cudaMemcpyAsync(Phi_body, dPhi, nb * 8, cudaMemcpyDeviceToHost, c->st));
        if (fx) PCE_CUDA(c, cudaMemcpyAsync(fx, dfx, N * 8, cudaMemcpyDeviceToHost, c->st));
        if (fy) PCE_CUDA(c, cudaMemcpyAsync(fy, dfy, N * 8, cudaMemcpyDeviceToHost, c->st));
        if (fz) PCE_CUDA(c, cudaMemcpyAsync(fz, dfz, N * 8, cudaMemcpyDeviceToHost, c->st));
        if (F && nb) PCE_CUDA(c, cudaMemcpyAsync(F, dF, 3 * nb * 8, cudaMemcpyDeviceToHost, c->st));
        if (T && nb) PCE_CUDA(c, cudaMemcpyAsync(T, dT, 3 * nb * 8, cudaMemcpyDeviceToHost, c->st));
        if (S && nb) PCE_CUDA(c, cudaMemcpyAsync(S, dS, 3 * nb * 8, cudaMemcpyDeviceToHost, c->st));
        if (U_tot) PCE_CUDA(c, cudaMemcpyAsync(U_tot, dU, 3 * 8, cudaMemcpyDeviceToHost, c->st));
        PCE_CUDA(c, cudaStreamSynchronize(c->st));
    }
    (void)tsave;
    timing_end(c);
    return rc ? rc : rc_solve;
}

// ---------------------------------------------------------------- reports
extern "C" int pce_set_timing(pce_ctx* c, int enabled)
{
    if (!c) return PCE_EINVAL;
    c->timing = enabled != 0;
    return PCE_OK;
}

extern "C" int pce_get_timings(const pce_ctx* c, pce_timings* t)
{
    if (!c || !t) return PCE_EINVAL;
    *t = c->tm;
    return PCE_OK;
}

extern "C" int pce_get_info(const pce_ctx* c, pce_info* info)
{
    if (!c || !info) return PCE_EINVAL;
    std::memset(info, 0, sizeof(*info));
    for (int d = 0; d < 3; ++d) {
        info->eta[d] = c->eta[d]; info->h[d] = c->h[d];
        info->ncell[d] = c->all.nc[d];
        info->image_range[d] = (c->all.nc[d] == 1) ? c->all.range[d] : 0;
    }
    info->nnz_near = c->nnz;
    info->N = c->N; info->N_bead = c->Nbead; info->N_body = c->Nbody;
    info->bytes_workspace = c->bytes;
    info->bytes_precond = c->pc_bytes;
    info->n_precond_blocks = c->pc_on ? c->pc_nblock : 0;
    info->P_matvec = c->P_mv;
    info->fft_mode = c->use_fftxy ? 2 : c->use_zfft ? 1 : 0;
    return PCE_OK;
}

extern "C" long long pce_launch_count(const pce_ctx* c) { return c ? c->launches : 0; }
