/*
 * pce.h -- C ABI of the B200 polarizable-colloid electrostatics library
 * (hot path of arxiv 2401.04865; citations are lines of the paper text,
 * "PAPER.md:N", with the equation they fall in).
 *
 * What the library computes
 * -------------------------
 * N particles (surface beads of N_body rigid conductors, then ions) of one
 * radius a in a triply periodic box.  The potential tensor (eq. 9)
 *     M_ab = 1/(eps_f V) sum_{k != 0} j0(ka)^2 exp(i k.(x_a-x_b)) / k^2
 * is applied by the spectral Ewald method of PAPER.md:167-268 (real-space sum
 * eq. 20-21, Gaussian spreading eq. 25, FFT, scaling eq. 26, inverse FFT,
 * Gaussian gather eq. 27), the induced bead charges follow from the
 * saddle-point system eq. 13 solved by a Krylov iteration on
 * the device, and energies / forces / torques from eqs. 14, 16-18
 * (PAPER.md:137-163).
 *
 * Conventions
 * -----------
 *  - every entry point returns 0 (PCE_OK) or a negative pce_status; no
 *    exception crosses the boundary; pce_last_error() gives the text.
 *  - "device" pointers are CUDA device memory of fp64 unless stated, owned by
 *    the CALLER (e.g. torch tensors), never retained past the call unless
 *    stated; "host" pointers are ordinary host memory.  The context owns all
 *    workspace (grids, cuFFT plans, cell lists, CSR near field, Krylov
 *    vectors) and frees it in pce_destroy.
 *  - all work is enqueued on the stream given to pce_create (a cudaStream_t
 *    passed as void*; NULL = default stream).  Calls are asynchronous except
 *    pce_solve (reads the residual) and pce_step_host.
 *  - particle order (structure of Sigma, eq. 52): beads of
 *    body 0, body 1, ... contiguous, then ions.  body_offset[N_body+1] (host,
 *    int32) gives the bead ranges; N_bead = body_offset[N_body].
 *  - SoA: x, y, z separate arrays.  Positions may lie outside [0,L); they
 *    are wrapped internally.  Results come back in caller order.
 *  - fp64 throughout.  There is no CPU fallback: without a CUDA device
 *    pce_create fails with PCE_ECUDA.
 */
#ifndef PCE_H
#define PCE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pce_ctx pce_ctx;

typedef enum {
    PCE_OK = 0,
    PCE_EINVAL = -1,   /* bad parameter / shape / NULL pointer */
    PCE_ENOMEM = -2,   /* device allocation failed */
    PCE_ECUDA = -3,    /* CUDA runtime error (text in pce_last_error) */
    PCE_ECUFFT = -4,   /* cuFFT plan / exec error */
    PCE_ENOCONV = -5,  /* Krylov solve hit max_iter; outputs still written */
    PCE_ESTATE = -6    /* call order violated (e.g. solve before set_system) */
} pce_status;

/* pce_params.flags */
#define PCE_FLAG_NO_PRECOND 1  /* plain (unpreconditioned) conjugate gradients in pce_solve */
#define PCE_FLAG_CUFFT_3D   2  /* 3-D cuFFT plans + separate scaling pass instead of 2-D cuFFT per plane + fused z pass */
#define PCE_FLAG_FIELD_IK   4  /* field mode of pce_evaluate / pce_forces: ik differentiation in wave space (E_d from the inverse
                                  transform of -i k_d times the scaled spectrum, gathered with the plain window: three more inverse
                                  transforms, wave-space momentum conserved to rounding) instead of the gradient of the gather
                                  window (default, one transform pair; reading A3). */

#define PCE_FLAG_DETERMINISTIC 8 /* bit-reproducible results: the gather writes one partial per (brick, particle) pair and adds each
                                  particle's partials in a fixed order instead of issuing fp64 atomics (the only run-to-run
                                  variation of the library, at the 1e-16 level); costs memory (8 B per pair and quantity) and
                                  ~15 % of the gather time.  Needs a mesh on the brick lattice (N_g % 8 == 0, N_g - P >= 8) */

/* Parameters of the spectral Ewald sum and of the solver.
 * eta is NOT a free input: eta = h^2 xi^2 P / pi (eq. 31,
 * PAPER.md:250), per dimension for a rectangular box. */
typedef struct {
    double L[3];        /* box edge lengths */
    int    Ng[3];       /* FFT grid nodes per dimension; each >= P */
    double xi;          /* Ewald splitting parameter, h(k)=exp(-k^2/4xi^2) */
    double rc;          /* real-space cut-off r_c (eq. 23); may exceed L/2 */
    int    P;           /* support grid points per dimension, even, 4..32 (eq. 29) */
    double a;           /* bead = ion radius: the shell regularization width (eq. 9-10) */
    double eps_f;       /* fluid permittivity (1 in the paper's units) */
    double tol_solver;  /* relative residual at which the Krylov solve stops */
    int    max_iter;    /* iteration cap of the Krylov solve */
    int    flags;       /* 0, or PCE_FLAG_* ORed */
    int    P_matvec;    /* support points per dimension of the SOLVER's bead-only matvec (pce_matvec, the Krylov iterations);
                           0 or P: the same window as everywhere (what pce_suggest_params sets).  The solver needs potentials
                           only, and at equal P the potential is ~5-20x more accurate than the window-gradient field, so
                           P - 2 keeps the induced charges within the tolerance (config 2: q error 5e-11 at P_matvec = 18,
                           tol 1e-10) and makes the spread / gather of every iteration (P_matvec / P)^3 = 0.73x as expensive
                           (config 5: step 184 -> 173 ms); the price is in ill-conditioned derived quantities -- the torque on
                           two nearly touching spheres (config 2, d = 2.2: a difference 1e5 times smaller than its terms)
                           moves from 7e-9 to 4e-8 relative.  Even, 4..P */
} pce_params;

typedef struct {
    int    iters;       /* Krylov iterations taken */
    int    matvecs;     /* applications of M inside pce_solve (bead-only + full) */
    double rel_resid;   /* final |P(b - M q)| / (|P r.E0|^2 + |P psi0|^2)^(1/2), psi0 = potential of the uniform starting
                           charges and the ions; a warm-started solve keeps the scale of the last cold solve if larger */
    int    converged;   /* 1 if rel_resid <= tol_solver */
    int    graph_replays; /* iterations enqueued as replays of the captured CUDA graph (0: plain kernel launches -- timing
                           enabled, PCE_NO_GRAPH=1, or a context on the legacy default stream, which cannot be captured) */
} pce_solve_info;

/* Per-pass device times (ms, CUDA events on the context's stream) summed over
 * the passes of the LAST pce_matvec / pce_evaluate / pce_solve / pce_forces
 * call that ran with timing enabled (pce_set_timing). */
typedef struct {
    double cells, real, spread, fft, scale, ifft, gather, krylov, other, total;
    /* the share of real / spread / gather spent in bead-only solver matvecs
     * (the rest belongs to full evaluations and the near-field build) */
    double bead_real, bead_spread, bead_gather;
    int    n_matvec_bead, n_eval_full, n_fft_pairs;
} pce_timings;

/* Derived quantities, for reports and tests. */
typedef struct {
    double eta[3], h[3];
    int    ncell[3];        /* real-space linked cells per dimension */
    int    image_range[3];  /* >0: periodic images summed explicitly in that dimension */
    long long nnz_near;     /* entries of the cached bead-bead near field */
    int    N, N_bead, N_body;
    long long bytes_workspace;
    long long bytes_precond; /* storage of the block-Jacobi preconditioner (bf16 for many large bodies, else fp32; 0: off) */
    int n_precond_blocks;    /* bodies that own a dense preconditioner block */
    int P_matvec;            /* support points per dimension of the solver's bead-only matvec */
    int fft_mode;            /* 0: cuFFT 3-D plans + scaling pass; 1: cuFFT 2-D per plane + fused z pass; 2: own (x, y) passes + fused z pass */
} pce_info;

/* Ewald parameters from a target tolerance (pure host arithmetic):
 * s^2 = -ln tol; k_c = pi (Ng-1)/L; xi = k_c/(2s) (eq. 28);
 * r_c = s/xi + 2a (eq. 23; the +2a because eq. 20 decays like
 * erfc((r-2a) xi) for shells, reading A14); P even with
 * exp(-pi P/2) a factor ~500 below tol (eq. 32), P_matvec = P.  P_override > 0 fixes P.
 * Fills L, Ng, xi, rc, P, P_matvec, a, eps_f=1, tol_solver=1e-12, max_iter=500. */
int pce_suggest_params(const double L[3], const int Ng[3], double a, double tol,
                       int P_override, pce_params* out);

/* Create a context on the current CUDA device.  `stream` is a cudaStream_t. */
int pce_create(const pce_params* p, void* stream, pce_ctx** out);
int pce_destroy(pce_ctx* ctx);
const char* pce_last_error(const pce_ctx* ctx); /* ctx may be NULL: last create error */

/* Declare the particle system and its positions (device x,y,z of length N).
 * body_offset: host int32[N_body+1], body_offset[0]=0, non-decreasing,
 * body_offset[N_body] = N_bead <= N.  Builds the linked cells,
 * body centres X_i (mean of the body's beads unwrapped about its first bead,
 * "centre of mass" PAPER.md:115) and r_ij = x_ij - X_i (eq. 12), and the
 * cached bead-bead real-space near field. */
int pce_set_system(pce_ctx* ctx, int N, int N_body, const int* body_offset,
                   const double* x, const double* y, const double* z);
/* New positions for the same system (e.g. next time step). */
int pce_set_positions(pce_ctx* ctx, const double* x, const double* y, const double* z);

/* Reference points X_i of the bodies (device X, Y, Z of length N_body) in place of the bead means: r_ij becomes the minimum
 * image of x_ij - X_i (eq. 12; the paper says "centre of mass").  The induced charges do not depend
 * on the choice (a shift d of X_i changes r_ij.E0 by a constant per body, absorbed by Phi_i -> Phi_i + d.E0); S_i, T_i, Psi_i
 * and U_i are then taken about the new point.  Valid until the next pce_set_positions / pce_set_system / pce_bd_step. */
int pce_set_centres(pce_ctx* ctx, const double* X, const double* Y, const double* Z);

/* psi = M_bb q over the N_bead conductor beads only (the solver's matvec;
 * eq. 8, restricted to bead sources and bead targets).
 * q, psi: device, length N_bead, caller order. */
int pce_matvec(pce_ctx* ctx, const double* q, double* psi);

/* Potentials psi_a - psi_0(x_a) = sum_b M_ab q_b (eq. 8 / eq. 19) and fields
 * E_a = -grad_a sum_b M_ab q_b (excludes E0; the b = a term has no gradient)
 * at all N particles from all N charges.  q, psi, Ex, Ey, Ez: device, length
 * N.  The three field pointers may all be NULL (potential only). */
int pce_evaluate(pce_ctx* ctx, const double* q, double* psi,
                 double* Ex, double* Ey, double* Ez);

/* Induced charges: eq. 13 with the ions as one-bead bodies of
 * fixed charge:  sum_j q_ij = Q_i  and
 * psi_ij - psi_0,ij = Phi_i + r_ij.E0,  Phi_i = Psi_i - Psi_0,i  (eq. 12).
 *  Q_body : device [N_body]; q_ion : device [N - N_bead] (may be NULL if no ions)
 *  E0     : host [3]
 *  q      : device [N]; out: bead charges then the ion charges.  If
 *           warm_start != 0 its bead part is read as the initial guess.
 *  Phi_body : device [N_body] out.
 * Method: conjugate gradients on the per-body-mean-projected SPD system,
 * whole iteration on the device, preconditioned (unless PCE_FLAG_NO_PRECOND)
 * by the inverse of each body's own free-space potential tensor (eq. 10) on
 * its zero-net-charge subspace.  That block depends on the body-frame bead
 * positions only, so it is built once in pce_set_system and stays valid while
 * pce_set_positions moves the bodies rigidly; a non-rigid
 * update costs iterations, never accuracy (the solution of eq. 13 is unique).
 * GMRES on the indefinite saddle-point form of eq. 13 (the paper's ref. 51 is GMRES-based) is not offered: M is
 * symmetric positive definite, the projected system is SPD, its solution is the unique solution of eq. 13, and
 * CG needs one vector of history and two fixed-order dot products per iteration where GMRES needs a growing basis.
 * Returns PCE_ENOCONV if max_iter was hit. */
int pce_solve(pce_ctx* ctx, const double* Q_body, const double* q_ion, const double E0[3],
              int warm_start, double* q, double* Phi_body, pce_solve_info* info);

/* Forces, torques, dipoles, energies for given charges q (device [N]):
 *  f_a = q_a (E0 + E_a)                               eq. 17
 *  F_i = sum_j f_ij,  T_i = sum_j r_ij x f_ij          eq. 18
 *  S_i = sum_j r_ij q_ij                               eq. 14
 *  U_i = (Q_i Psi_i - S_i.E0)/2, Psi_i = <psi_ij - r_ij.E0>_i - X_i.E0   eq. 16
 * Outputs (device; any may be NULL): fx,fy,fz [N]; F,T,S [3*N_body] as
 * (x[N_body], y[N_body], z[N_body]); U_body [N_body + N_ion] (ions:
 * q (psi - x.E0)/2); U_tot [3] = (U_eq16, W, U_MM) with U_MM = q.M.q/2 and
 * W = U_MM - sum_a q_a x_a.E0 (reading A8); psi [N] potentials. */
int pce_forces(pce_ctx* ctx, const double* q, const double E0[3],
               double* fx, double* fy, double* fz,
               double* F, double* T, double* S, double* U_body, double* U_tot, double* psi);

/* Grand capacitance tensor of the conductor bodies, C = Sigma' M^-1 Sigma'^T (eq. 15):
 *   [Q; S] = C [Psi - Psi_0; E_0],  blocks as in eq. 37.
 * M is the bead-bead potential tensor (eq. 9) of the N_bead conductor beads; ions are not conductors and are left out.
 * Index convention (Sigma' of the Appendix): k < N_body = potential / charge of body k;
 * k = N_body + 3 i + d = field / dipole component d of body i.  For every requested column k the SPD system
 * M_bb q = Sigma'^T e_k is solved on the device (conjugate gradients, preconditioned by the inverse of every body's own
 * free-space tensor) and its moments Sigma' q are returned.
 *  cols : host int[ncol], each in [0, 4 N_body);  C : device [ncol][4 N_body], row j = column cols[j] of C.
 * info (may be NULL): worst iteration count / residual over the columns, total matvecs.  PCE_ENOCONV if any column hit max_iter. */
int pce_capacitance_columns(pce_ctx* ctx, int ncol, const int* cols, double* C, pce_solve_info* info);

/* Effective permittivity tensor of the (periodic) dispersion, eq. 36:
 *   eps_eff = eps_f - n < C_SPsi C_qPsi^-1 C_qE - C_SE >,  n = N_body / V.
 * The bracket is the mean dipole response of floating bodies (Q = 0) to a field common to all bodies, so it is computed by
 * three constrained solves of eq. 13 with E0 = e_x, e_y, e_z, Q = 0 and no ionic charge (3 solves instead of 4 N_body
 * columns); the oracle evaluates eq. 36 from the blocks of C literally.  eps_eff: host [9], row-major. */
int pce_effective_permittivity(pce_ctx* ctx, double eps_eff[9], pce_solve_info* info);

/* Parameters of one Brownian-dynamics step. */
typedef struct {
    double dt;              /* time step (eq. 44) */
    double gamma;           /* Stokes drag coefficient of every ion and bead (eq. 43) */
    double kT;              /* thermal energy (eq. 41) */
    unsigned long long seed; /* key of the counter-based generator (used when `noise` is NULL) */
    unsigned int step;      /* time-step index: second counter word of the generator */
    int move_bodies;        /* 0: conductor bodies held fixed; 1: free-draining rigid-body motion (eq. 62) */
} pce_bd_params;

/* One Euler-Maruyama step of the overdamped Langevin equation (eqs. 40-44) from the context's current
 * positions, all on the device:
 *   hard spheres: eq. 46 as a pair potential at x(t): particles of different bodies closer than 2a repel
 *     with |f| = gamma (2a - r) / (2 dt), i.e. one step puts an overlapping pair back in contact; linked cells
 *     of edge >= 2a;
 *   ions: x += (f + f_hs) dt / gamma + sqrt(2 kT dt / gamma) N(0,1)  (eqs. 41-44).  N(0,1): `noise` (device, 3 N_ion doubles
 *     as x[N_ion], y[N_ion], z[N_ion]) or, if NULL, Philox-4x32-10 (counter = (ion index, step, 0, 0), key = seed) with
 *     Box-Muller on (r + 1/2) 2^-32: (sqrt(-2 ln u0) cos 2 pi u1, sqrt(-2 ln u0) sin 2 pi u1, sqrt(-2 ln u2) cos 2 pi u3);
 *   bodies (move_bodies): F_i, L_i of eq. 18 from f + f_hs, free-draining mobility (no hydrodynamic interactions,
 *     PAPER.md:382): U = F / (N_i gamma), Omega = [gamma sum_j (r_j^2 I - r_j r_j^T)]^-1 L, X += U dt, r_ij turned by the
 *     rotation exp([Omega dt]_x) (eq. 62 with U, Omega constant over the step); no Brownian displacement of bodies.
 * fx, fy, fz: device [N], the electrostatic forces of pce_forces (eq. 17).  The context then advances to the new positions
 * exactly as by pce_set_positions; x, y, z (device [N], may be NULL) receive them (wrapped into the box, caller order). */
int pce_bd_step(pce_ctx* ctx, const pce_bd_params* bp, const double* fx, const double* fy, const double* fz,
                const double* noise, double* x, double* y, double* z);

/* Double-layer observables about the centre of conductor body `body` from the context's current
 * positions and the charges q (device [N]): shells k = 0..n_bins-1 = [r_lo + k dr, r_lo + (k+1) dr), dr = 0.1 a
 * (PAPER.md:419), minimum-image distances of the IONS from the body centre.
 *   counts : device [2 n_bins]: cations (q > 0) then anions (q < 0) per shell ("shell summation")
 *   g      : device [2 n_bins]: eq. 49, count / (n_species * shell volume), n_species = N_species / V
 *   rho    : device [n_bins]: radial charge density, sliding window of width 2a about the shell midpoint
 *   Qcum   : device [n_bins]: eq. 48, Q + sum_{j<=k} rho_j dr, Q = net charge of the body's beads
 * Any output may be NULL. */
int pce_radial_profile(pce_ctx* ctx, int body, const double* q, double r_lo, int n_bins,
                       double* counts, double* g, double* rho, double* Qcum);

/* The same observables for a caller that must not allocate device memory -- an analysis hook inside a simulation engine
 * whose own pool has claimed the GPU's memory (so a cudaMalloc may fail in the middle of a run), or one that runs between the
 * engine's kernels, where cudaMalloc / cudaFree would stall the whole device.  No pce_ctx is needed and the call makes no
 * cudaMalloc, cudaFree or allocating library call: its one scratch buffer, the integer shell counters, is a fixed
 * 128 KiB array inside the library image (held by every GPU that loads libpce.so until the process exits).
 *   stream  : cudaStream_t the work is enqueued on (NULL: default stream); the call does not wait for it
 *   x, y, z, q_ion : device [n_ion], positions (anywhere; minimum image is taken) and charges of the IONS only
 *   q_bead  : device [n_bead], charges of the beads of the body the profile is taken about (Q of eq. 48 is their sum;
 *             n_bead = 0: Q = 0)
 *   centre, L : host [3], the body's reference point X_i and the box edges;  a: particle radius, dr = 0.1 a
 *   counts, g, rho, Qcum : device, as in pce_radial_profile, owned by the caller; any may be NULL, Qcum needs rho
 *   err     : host buffer of err_len bytes (may be NULL) that receives the text of a failure
 * Limit: n_bins <= PCE_PROFILE_STATIC_MAX_BINS; more is refused with PCE_EINVAL (split [r_lo, r_hi) over several calls --
 * counts, g and rho of a shell do not depend on the other shells; only Qcum carries the running sum).
 * Set-up: the first call made with a given device current looks up the device address of the counter array
 * (cudaGetSymbolAddress, once per device, under a lock); make that first call before any stream capture is begun.
 * Sharing: every call on a device uses the same counters.  Each call zeroes the part it uses on `stream` before binning, so
 * calls enqueued one after another on one stream are independent; two calls that can overlap on the GPU (different streams,
 * different host threads without ordering between them) race on the counters and both results are garbage. */
#define PCE_PROFILE_STATIC_MAX_BINS 16384
int pce_radial_profile_static(void* stream, int n_ion, const double* x, const double* y, const double* z, const double* q_ion,
                              int n_bead, const double* q_bead, const double centre[3], const double L[3], double a,
                              double r_lo, int n_bins, double* counts, double* g, double* rho, double* Qcum,
                              char* err, int err_len);

/* One whole pass of the hot path from HOST buffers (what bench.py's "e2e"
 * times): copy positions and charges to the device, rebuild cells, solve
 * eq. 13, evaluate forces, copy results back.  All pointers host; x,y,z [N];
 * outputs as in pce_solve / pce_forces (any output may be NULL).  warm_start != 0: the bead part of q (host, [N]) is
 * read as the initial guess of the solve (e.g. the charges of the previous time step), as in pce_solve. */
int pce_step_host(pce_ctx* ctx, const double* x, const double* y, const double* z,
                  const double* Q_body, const double* q_ion, const double E0[3], int warm_start,
                  double* q, double* Phi_body, double* fx, double* fy, double* fz,
                  double* F, double* T, double* S, double* U_tot, pce_solve_info* info);

/* Host-only test hook (no GPU needed): the real-space pair kernel R(r) (eq. 20) and dR/dr exactly as
 * the device evaluates them -- piecewise degree-7 polynomials in r^2 of the six exp/erfc terms plus the closed-form
 * Heaviside term -- for n radii r[i] in [a/4, r_c); entries outside that range come back NaN (the device uses the
 * exact formula there).  All pointers host. */
int pce_real_kernel_host(double a, double xi, double rc, double eps_f, int n, const double* r, double* R, double* dR);

/* Measured fp64 roofs of the current device (register-resident chains, ~10 ms): tflops[0] = DFMA on the vector pipe,
 * tflops[1] = mma.sync.m8n8k4.f64 on the tensor path.  Host pointer.  bench.py reports the spread / gather passes against them. */
int pce_measure_fp64_peaks(double tflops[2]);

/* Test hook: overwrite the shared memory of every SM with NaN bit patterns (on `stream`, a cudaStream_t), so that a kernel
 * reading shared memory it never wrote poisons its result visibly.  No effect on any context. */
int pce_debug_poison_shared_memory(void* stream);

int pce_set_timing(pce_ctx* ctx, int enabled);          /* per-pass CUDA events on/off (default off) */
int pce_get_timings(const pce_ctx* ctx, pce_timings* t);
int pce_get_info(const pce_ctx* ctx, pce_info* info);
/* number of kernels of this library (cuFFT's own excluded) launched since create */
long long pce_launch_count(const pce_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* PCE_H */
