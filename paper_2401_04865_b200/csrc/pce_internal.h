// pce_internal.h -- shared declarations of the CUDA implementation (not part of the ABI).
// Product code: never includes or links anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "pce.h"
#include "realtab.h"

#define PCE_PI 3.14159265358979323846

// 64-byte hit record of one particle for the cached-list spread / gather (wave_cols.cu): per dimension the two coefficients
// (c_m, e1) of the exp-free window recurrence -- c_m = exp(-aw u0 (u0 + 2 (phi - 8))), the weight factor at support index
// phi - 8, and e1 = exp(-2 aw u0) --, the first support index per dimension (int16: meshes up to 32767) and the charge
struct alignas(16) HitRec {
    double2 cf[3];
    short s0[3], pad;
    double q;
};
static_assert(sizeof(HitRec) == 64, "hit records are 64 bytes");
constexpr int HITREC_Q_STRIDE = sizeof(HitRec) / sizeof(double);  // doubles between the charges of consecutive records

// ---------------------------------------------------------------- binning
// A counting-sort binning of a particle subset into a Cartesian cell grid
// (linked-cell neighbour search).  In a dimension with fewer
// than 3 cells of size >= r_c the grid collapses to ONE cell and periodic
// images -range..range are summed explicitly (covers r_c > L/2).
struct Bins {
    int n = 0;          // particles in the subset
    int nc[3] = {1, 1, 1};
    int ncell = 1;
    int range[3] = {1, 1, 1};  // stencil half width: 1 (cells) or image count
    double L[3];
    // cell index per dimension = min(((min((int)(x * scale), imax) + shift) mod (imax + 1)) / div, nc - 1):
    //   real-space cells: scale = nc/L, div = 1, shift = 0;
    //   mesh bins: scale = 1/h, imax = Ng-1, div = brick edge, shift = P/2 mod brick edge
    double scale[3] = {1, 1, 1};
    int imax[3] = {0, 0, 0}, div[3] = {1, 1, 1}, shift[3] = {0, 0, 0};
    int* inv = nullptr;         // [n] index in the subset -> sorted slot
    int* cell_of = nullptr;     // [n]
    int* cell_start = nullptr;  // [ncell+1]
    int* cell_fill = nullptr;   // [ncell+1] scratch
    int* chunk_start = nullptr; // [ncell+1] real-space binnings: first 32-target chunk of each cell (scan of ceil(n_cell/32))
    int* perm = nullptr;        // [n] sorted slot -> index in the subset
    int* perm_tmp = nullptr;    // [n]
    double *xs = nullptr, *ys = nullptr, *zs = nullptr;  // [n] sorted, wrapped
    double* qs = nullptr;                                // [n] sorted charges (per call)
    // mesh binnings only: per-particle window coefficients (wave_bricks.cu, k_window_coef)
    int4* ws0 = nullptr;      // [n] first support mesh index per dimension (x, y, z, unused)
    double4* wcf = nullptr;   // [3 n] per particle and dimension: (c0, e1, e8, 1/e8), see wave_bricks.cu
    // mesh binnings on brick-aligned meshes: cached hit lists (wave_cols.cu)
    HitRec* hrec = nullptr;       // [n]
    double4* wu0 = nullptr;       // [n] (u0x, u0y, u0z, -): offset of the first support point from the particle, mesh units
    int* col_cnt = nullptr;       // [nkeys + 1] key counters (build), then the list of crowded keys
    int* col_start = nullptr;     // [nkeys + 1] first entry of key (column, z_k)
    int* col_ent = nullptr;       // [col_ent_cap] particle slots ordered by (column, z_k, slot)
    int* item_start = nullptr;    // [ncell + 1] first work item of each brick (chunked binnings)
    int2* items = nullptr;        // [col_item_cap] (brick, chunk)
    double* col_scratch = nullptr;  // [col_item_cap][512] partial bricks of split bricks
    int* col_arrive = nullptr;    // [ncell] arrival counters of split bricks
    double* qs_cols = nullptr;    // &hrec[0].q: charges are written into the records (stride HITREC_Q_STRIDE doubles)
    int col_chunk = 0, n_items = 0;
    // deterministic gather (PCE_FLAG_DETERMINISTIC): pair numbering per brick, per-particle pair lists
    int* pair_start = nullptr;    // [ncell + 1]
    int* inv_ptr = nullptr;       // [n + 1]
    int* inv_list = nullptr;      // [inv_cap] pair ids of each particle in a fixed order
    int n_pairs = 0;
    long long inv_cap = 0;
    long long col_ent_cap = 0, col_item_cap = 0, nkeys = 0;
};

// real-space kernel constants (eq. 20/21)
struct RealConst {
    double a, xi, two_a, c64, rc2, R0, inv_eps;
    double two_xi_sqrtpi;   // 2 xi / sqrt(pi)
    double t_lin, t_quad;   // small-r Taylor: R ~ R0 - t_lin r + t_quad r^2
    double r_small;         // below this the Taylor form is used
};

// wave-space constants (eq. 25-27)
struct WaveConst {
    int Ng[3];
    int Nxh;            // Ng[0]/2+1
    int P;
    double L[3], h[3], inv_h[3];
    double aw;          // Gaussian exponent in grid units: exp(-aw u^2), aw = 2 pi / P
    double kfac[3];     // 2 pi / L_d
    double gexp[3];     // (1-eta_d)/(4 xi^2)
    double a;           // bead radius (shape factor j0(ka))
    double scale_norm;  // c_n^2 h^3 / (eps N_tot)
    double grad_fac[3]; // 2 alpha_w,d h_d = 4 pi /(P h_d): dW/dx_alpha = grad_fac * u * W
    double G[32];       // exp(-aw r^2), r = 0..P-1
};

// Device-resident state of the Krylov solve (krylov.cu): every step length, the stopping test and the iteration count live
// here; the host only watches CgHostStatus.
struct CgState {
    double rz[2];        // g.z of the current iteration at [it & 1] (the previous one at the other slot)
    double pap, gg;      // p.Ap, |g|^2
    double psum;         // sum of the search direction (k = 0 constant of the operator, reading A1)
    double ref, ref_cold;  // residual scale; the one of the last cold-start solve
    double ref_saved;      // ref_cold of the caller's solves while pce_effective_permittivity runs its own
    double tol;
    int it, maxit, done, project;  // project = 1: eq. 13 on the per-body-mean-projected subspace; 0: plain M q = b
    unsigned cnt[8];     // arrival counters of the last-block-done reductions
};
struct CgHostStatus {
    volatile int it, done;
    volatile double gg, ref;
};

enum Pass { PASS_CELLS = 0, PASS_REAL, PASS_SPREAD, PASS_FFT, PASS_SCALE, PASS_IFFT, PASS_GATHER, PASS_KRYLOV, PASS_OTHER, PASS_COUNT };

struct pce_ctx {
    pce_params p;
    cudaStream_t st = nullptr;
    std::string err;
    RealConst rk;
    RealTable rt;              // real-space kernel table (device pointer), realtab.h
    double* rt_dev = nullptr;
    WaveConst wk;              // the ACTIVE wave-space constants (wave_select): a copy of wset[0] or wset[1]
    WaveConst wset[2];         // [0]: window of P points (evaluations, right-hand side); [1]: P_matvec points (solver matvec)
    int P_mv = 0;              // = P_matvec (or P)
    double V = 0, eta[3], h[3];
    double kconst = 0;  // 1/(4 xi^2 V eps)

    int N = 0, Nbead = 0, Nbody = 0, Nion = 0;
    bool have_system = false;
    std::vector<int> body_off_h;

    double *x = nullptr, *y = nullptr, *z = nullptr;     // [N] wrapped, caller order
    int* body_off = nullptr;                             // [Nbody+1]
    int* body_of = nullptr;                              // [Nbead]
    double *rx = nullptr, *ry = nullptr, *rz = nullptr;  // [Nbead] r_ij
    double *X = nullptr, *Y = nullptr, *Z = nullptr;     // [Nbody] centres (unwrapped about first bead)

    Bins all, bead;    // real-space linked cells (all particles / conductor beads)
    Bins wall, wbead;  // mesh tiles (spread / gather), window of P points
    Bins wbead_s;      // the beads binned for the window of P_matvec points (only if P_matvec != P)
    Bins* wmv = nullptr;  // the bead binning of the solver matvec: &wbead_s or &wbead
    int* scan_tmp = nullptr;  // block sums for the scans
    size_t scan_tmp_n = 0;

    // cached bead-bead near field (CSR over the bead binning's sorted order)
    int* csr_ptr = nullptr;
    int* csr_col = nullptr;
    double* csr_val = nullptr;
    long long nnz = 0, nnz_cap = 0;

    // mesh
    double* grid = nullptr;
    cufftDoubleComplex* gridk = nullptr;
    cufftDoubleComplex* gridk2 = nullptr;  // second half spectrum (ik-differentiated fields: the forward spectrum is used four times)
    cufftHandle planF = 0, planB = 0;
    void* fft_work = nullptr;
    bool have_plans = false;
    bool use_zfft = false;     // 2-D cuFFT per plane + fused z FFT / Green's function / inverse z FFT (zfft.cu)
    double2* ztw = nullptr;    // twiddles exp(-2 pi i m / N_z)
    double* zexp = nullptr;    // per-axis Gaussian factors of the Green's function (active set)
    double* zexp_set[2] = {nullptr, nullptr};
    double* zshape = nullptr;  // piecewise-polynomial table of the shape factor j0(ka)^2 / k^2 as a function of k^2
    int zshape_key_lo = 0, zshape_n = 0;
    bool use_fftxy = false;    // own (x, y) transforms, one HBM trip per plane and direction (fftxy.cu) instead of cuFFT 2-D plans
    double2* xytw = nullptr;   // twiddles exp(-2 pi i m / N_x)
    int* xy_ctr = nullptr;     // [1 + N_z] work counter + per-plane arrival counters
    int xy_occ[2] = {0, 0}, xy_nt[2] = {128, 128};  // per direction (forward, inverse): resident CTAs per SM, threads per CTA
    bool zfft_attr_set = false;  // dynamic shared-memory limit of k_zfft_scale raised on this context's device
    // persistent brick kernels (wave_bricks.cu)
    int num_sm = 0, occ_spread = 0, occ_gather = 0, occ_gather_f = 0;
    bool use_cols = false;     // cached-list spread / gather (wave_cols.cu) instead of the per-call candidate walk
    int occ_cspread = 0, occ_cgather = 0, occ_cgather_f = 0;
    int* work_ctr = nullptr;
    double* gather_part = nullptr;  // per-(brick, hit) partial sums of the deterministic gather
    long long part_cap = 0;

    // per-call work vectors
    double *w_real = nullptr, *w_wave = nullptr;            // [N] sorted-order potentials
    double *w_ex = nullptr, *w_ey = nullptr, *w_ez = nullptr;  // [N] sorted-order real-space field
    double *w_kx = nullptr, *w_ky = nullptr, *w_kz = nullptr;  // [N] sorted-order wave-space field
    double* scal = nullptr;  // device scalars
    double* sum_part = nullptr;  // [1024] partial sums
    // Krylov vectors [Nbead]
    double *cg_g = nullptr, *cg_p = nullptr, *cg_t = nullptr, *cg_ap = nullptr, *cg_psi = nullptr;
    double *ev_psi = nullptr, *ev_ex = nullptr, *ev_ey = nullptr, *ev_ez = nullptr;  // [N]
    double* cg_q = nullptr;     // [Nbead] the iterate (copied to the caller's array when the solve ends)
    double* cg_part = nullptr;  // [3 * max(Nbody, pupdate blocks)] per-block partials of the fixed-order sums
    CgState* cg_state = nullptr;        // device
    CgHostStatus* cg_host = nullptr;    // pinned, mapped: progress of the solve as the device reports it
    CgHostStatus* cg_host_dev = nullptr;  // its device address
    cudaGraphExec_t cg_graph = nullptr; // one captured Krylov iteration (matvec + vector kernels)
    bool cg_graph_failed = false;
    bool cg_graph_stale = false;        // positions / a buffer the graph names changed: capture again before the next replay
    long long cg_graph_launches = 0;    // kernels of this library inside one replay
    const int* skip_flag = nullptr;     // when set, the operator kernels return at once if *skip_flag != 0 (solver converged)
    // block-Jacobi preconditioner (precond.cu)
    bool pc_on = false;
    void* pc_B = nullptr;             // per-body n_i x n_i blocks in bf16 or fp32, rows padded to 8 entries
    bool pc_bf16 = false;
    void* pc_rows = nullptr;          // CTA -> (body, first row) map of the apply kernel
    unsigned char* pc_has = nullptr;  // [Nbody] 1 if the body has a dense block
    int pc_nrows_cta = 0, pc_max_n = 0, pc_nblock = 0;
    long long pc_bytes = 0;
    double* cg_z = nullptr;           // [Nbead] B r before the mean is removed
    double* pc_mean = nullptr;        // [Nbody]
    double* pc_u = nullptr;           // [Nbead] u = A^-1 1 of each body's block (0: no block)
    double* pc_invs = nullptr;        // [Nbody] 1 / (1.u)
    // Brownian dynamics (dynamics.cu): linked cells of edge >= 2a, hard-sphere forces, the new positions, profile counters
    Bins hs;
    bool hs_ready = false;
    double *bd_f = nullptr;   // [3 N] hard-sphere forces, caller order (x | y | z)
    double *bd_x = nullptr;   // [3 N] new positions (x | y | z)
    unsigned* prof_cnt = nullptr;  // [2 n_bins] shell counts
    int prof_cnt_n = 0;
    // host staging for pce_step_host
    double* hs_dev = nullptr;
    size_t hs_dev_n = 0;

    long long bytes = 0;
    long long bytes_base = 0;  // workspace that survives free_system (grids, plans, tables)
    long long launches = 0;

    // timing
    bool timing = false;
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    struct Rec { int pass; bool bead; cudaEvent_t a, b; };
    bool in_bead_matvec = false;
    std::vector<Rec> recs;
    pce_timings tm;
};

// ---------------------------------------------------------------- helpers
#define PCE_CUDA(ctx, call)                                                            \
    do {                                                                               \
        cudaError_t e__ = (call);                                                      \
        if (e__ != cudaSuccess) {                                                      \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);           \
            return PCE_ECUDA;                                                          \
        }                                                                              \
    } while (0)

static inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

struct PassTimer {
    pce_ctx* c;
    int pass;
    cudaEvent_t a = nullptr, b = nullptr;
    PassTimer(pce_ctx* ctx, int pass_) : c(ctx), pass(pass_) {
        if (!c->timing) return;
        while (c->ev_used + 2 > c->ev_pool.size()) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            c->ev_pool.push_back(e);
        }
        a = c->ev_pool[c->ev_used++];
        b = c->ev_pool[c->ev_used++];
        cudaEventRecord(a, c->st);
    }
    ~PassTimer() {
        if (!c->timing) return;
        cudaEventRecord(b, c->st);
        c->recs.push_back({pass, c->in_bead_matvec, a, b});
    }
};

// cells.cu
int bins_alloc(pce_ctx* c, Bins& b, int n, const int nc[3], const int range[3]);          // real-space cells
int bins_alloc_chunks(pce_ctx* c, Bins& b);
int bins_alloc_tiles(pce_ctx* c, Bins& b, int n, int tile);                                  // mesh tiles of `tile` grid points
void bins_free(Bins& b);
int bins_build(pce_ctx* c, Bins& b, const double* x, const double* y, const double* z);
int exclusive_scan(pce_ctx* c, int* data, int n_plus_1);  // in place over n+1 entries (last input must be 0)
int wrap_positions(pce_ctx* c, int n, const double* xi, const double* yi, const double* zi, double* xo, double* yo, double* zo);
int gather_by_perm(pce_ctx* c, int n, const int* perm, const double* in, double* out, int out_stride = 1);

// realspace.cu
int real_direct(pce_ctx* c, const Bins& tb, const Bins& sb, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s);
int real_csr_build(pce_ctx* c, const Bins& b);
int real_csr_spmv(pce_ctx* c, const Bins& b, double* psi_s);

// realtab.cu
void realtab_build_host(double a, double xi, double rc, std::vector<double>& tab, RealTable& T);
int realtab_upload(pce_ctx* c);
void chebtab_build(double s_lo, double s_hi, long double (*f)(long double, const void*), const void* ctx, std::vector<double>& tab,
                   int& key_lo, int& n_int);

// pce_api.cu
void wave_select(pce_ctx* c, int which);  // 0: window of P points, 1: window of P_matvec points (solver matvec)

// wave.cu
int wave_fft_scale_ifft(pce_ctx* c);
int wave_forward(pce_ctx* c);                 // mesh -> (x, y)-transformed half spectrum (or the full 3-D transform)
int wave_scale_inverse(pce_ctx* c, int deriv);  // Green's function (times -i k_d if deriv >= 0) and back to the mesh; the forward spectrum is kept when deriv >= 0

// zfft.cu
bool zfft_supported(const pce_params& p);
int zfft_init(pce_ctx* c);
int zfft_scale(pce_ctx* c, const void* in, void* out, int deriv);  // deriv = -1: potential; 0..2: times -i k_d (field component d)

// fftxy.cu
bool fftxy_supported(const pce_params& p);
int fftxy_init(pce_ctx* c);
int fftxy_forward(pce_ctx* c, cufftDoubleComplex* gk);   // c->grid -> gk (x, y transformed, plane by plane)
int fftxy_inverse(pce_ctx* c, cufftDoubleComplex* gk);   // gk -> c->grid

// wave_bricks.cu
int wave_bricks_init(pce_ctx* c);
int wave_coef_alloc(pce_ctx* c, Bins& b);
int wave_window_coef(pce_ctx* c, const Bins& b);
int wave_spread_bricks(pce_ctx* c, const Bins& b);
int wave_gather_bricks(pce_ctx* c, const Bins& b, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s);

// wave_cols.cu
bool wave_cols_supported(const pce_ctx* c);
int wave_cols_init(pce_ctx* c);
int wave_cols_alloc(pce_ctx* c, Bins& b);
void wave_cols_free(Bins& b);
int wave_cols_build(pce_ctx* c, Bins& b);
int wave_spread_cols(pce_ctx* c, const Bins& b);
int wave_gather_cols(pce_ctx* c, const Bins& b, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s);

// krylov.cu
int bodies_setup(pce_ctx* c);
int bodies_set_centres(pce_ctx* c, const double* X, const double* Y, const double* Z);
int solve_cg(pce_ctx* c, const double* Q_body, const double* q_ion, const double E0[3], int warm, double* q, double* Phi, pce_solve_info* info);
int solve_plain(pce_ctx* c, const double* b, double* q, pce_solve_info* info);  // M_bb q = b (no constraint), b and q device [Nbead]
int capacitance_columns(pce_ctx* c, int ncol, const int* cols, double* C, pce_solve_info* info);
int effective_permittivity(pce_ctx* c, double eps_eff[9], pce_solve_info* info);
void krylov_free(pce_ctx* c);
void krylov_invalidate_graph(pce_ctx* c);
// per-call timing records (pce_api.cu): every entry point that opens PassTimers brackets itself with these
void timing_begin(pce_ctx* c);
void timing_end(pce_ctx* c);
struct TimingScope {
    pce_ctx* c;
    explicit TimingScope(pce_ctx* c_) : c(c_) { timing_begin(c); }
    ~TimingScope() { timing_end(c); }
};
int op_matvec_bead_sorted(pce_ctx* c);  // sorted charges in bead.qs / wbead.qs -> w_real / w_wave (sorted orders)
int forces_all(pce_ctx* c, const double* q, const double E0[3], double* fx, double* fy, double* fz, double* F, double* T,
               double* S, double* U_body, double* U_tot, double* psi_out);

// dynamics.cu
void dynamics_free(pce_ctx* c);
int positions_update(pce_ctx* c, const double* x, const double* y, const double* z);  // pce_api.cu: what pce_set_positions does

// precond.cu
int precond_setup(pce_ctx* c);
void precond_free(pce_ctx* c);
int precond_apply(pce_ctx* c, const double* r, double* z);

// pce_api.cu
int sum_vector(pce_ctx* c, const double* in, int n, double* out);  // deterministic two-stage sum
int op_matvec_bead(pce_ctx* c, const double* q, double* psi);
int op_evaluate(pce_ctx* c, const double* q, double* psi, double* Ex, double* Ey, double* Ez);
int op_evaluate_at_beads(pce_ctx* c, const double* q, double* psi);
