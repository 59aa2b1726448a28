// realspace.cu -- real-space part of the Ewald split (eq. 19 second line):
// the closed-form pair kernel eq. 20, its r -> 0 limit
// eq. 21 and its derivative (not printed in the paper; derived
// in DESIGN.md "Real-space kernel"), summed over linked-cell neighbours
// (PAPER.md:200, 262).  Two uses: a direct pass (potential, optionally field)
// and a cached CSR near field for the bead-only solver matvec, positions
// being frozen during a Krylov solve.
#include "pce_internal.h"

struct CellGeom {
    int nc[3], range[3];
    double L[3], inv_cell[3];
};

static CellGeom geom_of(const Bins& b)
{
    CellGeom g;
    for (int d = 0; d < 3; ++d) {
        g.nc[d] = b.nc[d]; g.range[d] = b.range[d]; g.L[d] = b.L[d]; g.inv_cell[d] = b.nc[d] / b.L[d];
    }
    return g;
}

// F(u) = (2 xi^2 u^2 + 1) erfc(u xi) - (2 xi/sqrt(pi)) u exp(-u^2 xi^2), u >= 0.
// eq. 20's six exp/erfc terms are c64/r [F(r+2a) + F(r-2a) - 2F(r)], c64 = 1/(64 pi a^2 xi^2);
// for r < 2a, F(r-2a) = 2(2 xi^2 (r-2a)^2 + 1) - F(2a-r) and the polynomial part
// cancels the Heaviside term up to 2 c64 / r.
__device__ __forceinline__ void F_and_dF(double u, double xi, double& F, double& dF)
{
    const double x = u * xi;
    const double e = exp(-x * x);
    const double ecx = erfcx(x);
    const double isp = 0.56418958354775628695;  // 1/sqrt(pi)
    F = e * ((2.0 * x * x + 1.0) * ecx - 2.0 * isp * x);
    dF = xi * e * (4.0 * x * ecx - 4.0 * isp);
}

// R(r) and dR/dr for r > 0 (times eps_f)
__device__ __forceinline__ void pair_kernel(const RealConst& k, double r, double& R, double& dR)
{
    if (r < k.r_small) {
        R = k.R0 - k.t_lin * r + k.t_quad * r * r;
        dR = -k.t_lin + 2.0 * k.t_quad * r;
        return;
    }
    double Fp, dFp, Fm, dFm, Fr, dFr;
    F_and_dF(r + k.two_a, k.xi, Fp, dFp);
    F_and_dF(fabs(r - k.two_a), k.xi, Fm, dFm);
    F_and_dF(r, k.xi, Fr, dFr);
    const double B = (r >= k.two_a) ? (Fp + Fm - 2.0 * Fr) : (Fp - Fm - 2.0 * Fr + 2.0);
    const double dB = dFp + dFm - 2.0 * dFr;
    const double ir = 1.0 / r;
    R = k.c64 * B * ir;
    dR = k.c64 * ir * (dB - B * ir);
}

__device__ __forceinline__ int floor_div(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

// visit every (neighbour j, image) of sorted particle i with r < r_c
template <class Op>
__device__ __forceinline__ void for_neighbors(const CellGeom& g, const int* __restrict__ cell_start, const double* __restrict__ xs,
                                              const double* __restrict__ ys, const double* __restrict__ zs, int i, double rc2, Op& op)
{
    const double xi = xs[i], yi = ys[i], zi = zs[i];
    const int cx = min((int)(xi * g.inv_cell[0]), g.nc[0] - 1);
    const int cy = min((int)(yi * g.inv_cell[1]), g.nc[1] - 1);
    const int cz = min((int)(zi * g.inv_cell[2]), g.nc[2] - 1);
    for (int oz = -g.range[2]; oz <= g.range[2]; ++oz) {
        int nz = cz + oz;
        const int wz = floor_div(nz, g.nc[2]);
        nz -= wz * g.nc[2];
        const double sz = wz * g.L[2];
        for (int oy = -g.range[1]; oy <= g.range[1]; ++oy) {
            int ny = cy + oy;
            const int wy = floor_div(ny, g.nc[1]);
            ny -= wy * g.nc[1];
            const double sy = wy * g.L[1];
            for (int ox = -g.range[0]; ox <= g.range[0]; ++ox) {
                int nx = cx + ox;
                const int wx = floor_div(nx, g.nc[0]);
                nx -= wx * g.nc[0];
                const double sx = wx * g.L[0];
                const int cell = (nz * g.nc[1] + ny) * g.nc[0] + nx;
                const int jb = cell_start[cell], je = cell_start[cell + 1];
                const bool home = (ox == 0 && oy == 0 && oz == 0);
                for (int j = jb; j < je; ++j) {
                    if (home && j == i) continue;  // beta = alpha, n = 0: the self term (eq. 21)
                    const double dx = xi - (xs[j] + sx), dy = yi - (ys[j] + sy), dz = zi - (zs[j] + sz);
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    if (r2 < rc2) op(j, dx, dy, dz, r2);
                }
            }
        }
    }
}

// R(r) and g = -R'(r)/r (times eps_f) at s = r^2 > 0: table of realtab.h + closed-form Heaviside term; exact below s_lo
template <int NS = 0>
__device__ __forceinline__ void pair_eval(const RealConst& k, const RealTable& T, double s, bool field, double& R, double& g,
                                          const double* sh = nullptr)
{
    if (s >= T.s_lo) {
        if (NS > 0) rt_eval_sh<NS>(sh, T.key_lo, s, field, R, g);
        else rt_eval(T, s, field, R, g);
        if (s < k.two_a * k.two_a) {  // overlapping shells: Heaviside term of eq. 20 (reading G3)
            const double ir = rsqrt(s), r = s * ir, m = r - k.two_a;
            R -= m * m * k.t_lin * ir;                                      // t_lin = 1/(16 pi a^2)
            g -= (0.25 / PCE_PI * ir * ir - k.t_lin) * ir;
        }
    } else {
        const double r = sqrt(s);
        double dR;
        pair_kernel(k, r, R, dR);
        g = -dR / r;
    }
}

// ---------------------------------------------------------------- direct pass (step 1)
// The paper runs one thread per particle over the neighbour cells.  Here one WARP owns a chunk of up to 32 targets of one
// cell (persistent warps, chunks handed out by a global counter): lane l owns target l, the sources of each of the 27 neighbour cells (or periodic images, reading A10) are
// staged 64 at a time in the warp's shared memory by coalesced loads, every lane tests its target against the 64
// staged sources (broadcast reads, 7 fp64 instructions per test) and records the hits in a 64-bit mask; the kernel
// (two degree-7 polynomials from the table) is then evaluated hit by hit, so the expensive body runs max_lane(hits)
// times per stage instead of once per candidate.  Targets and sources may be different subsets with the same cell
// geometry (targets = beads, sources = all, for the right-hand side of eq. 13).  A source at r = 0 -- the target
// itself (the beta = alpha, n = 0 term) or a coincident particle (reading A9) -- contributes R(0) q (eq. 21) and no field.
constexpr int RS_WARPS = 4;        // warps per CTA, a chunk per warp
constexpr int RS_SPLIT_WARPS = 8;  // warps per CTA when the CTA shares one chunk (small systems)
constexpr int RS_STAGE = 64;

// SPLIT = 1: a warp per chunk.  SPLIT = WARPS (few chunks: small systems, where one warp walking ~1000 candidates per target is
// the critical path of the whole launch): the CTA owns the chunk, warp w takes every WARPS-th source stage, the partial sums
// are added in warp order (deterministic).
// NS > 0: the table sits in shared memory with the compile-time row stride NS (realtab.h); NS = 0: global memory, generic loads.
template <bool FIELD, int WARPS, int SPLIT, int NS>
__global__ void __launch_bounds__(WARPS * 32)
k_real_cells(CellGeom g, RealConst k, RealTable T, const int* __restrict__ t_start, const int* __restrict__ t_chunk,
             const double* __restrict__ txs,
             const double* __restrict__ tys, const double* __restrict__ tzs, const int* __restrict__ s_start,
             const double* __restrict__ sxs, const double* __restrict__ sys, const double* __restrict__ szs,
             const double* __restrict__ sqs, double* __restrict__ psi, double* __restrict__ ex, double* __restrict__ ey,
             double* __restrict__ ez, int* __restrict__ work_ctr)
{
    __shared__ double2 sh_xy[WARPS][RS_STAGE];
    __shared__ double2 sh_zq[WARPS][RS_STAGE];
    extern __shared__ double sh_tab[];  // copy of the kernel table (potential rows, with FIELD also the field rows), row stride NS
    if (NS > 0) {
        constexpr int rows = FIELD ? RT_STRIDE : RT_DEG + 1;
        for (int e = threadIdx.x; e < rows * T.n_int; e += blockDim.x) sh_tab[(e / T.n_int) * NS + e % T.n_int] = T.tab[e];
        __syncthreads();
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double2* sxy = sh_xy[warp];
    double2* szq = sh_zq[warp];
    __shared__ int sh_item;
    __shared__ double sh_part[SPLIT > 1 ? WARPS : 1][4][32];
    const int ncell = g.nc[0] * g.nc[1] * g.nc[2];
    for (;;) {
        // work item: one chunk of up to 32 targets of ONE cell (cells.cu scans ceil(n_cell/32) into t_chunk): a crowded cell
        // is shared by many warps, a warp never straddles cells
        int item = 0;
        if (SPLIT > 1) {
            __syncthreads();  // the previous item's partial sums are consumed
            if (threadIdx.x == 0) sh_item = atomicAdd(work_ctr, 1);
            __syncthreads();
            item = sh_item;
        } else {
            if (lane == 0) item = atomicAdd(work_ctr, 1);
            item = __shfl_sync(0xffffffffu, item, 0);
        }
        if (item >= t_chunk[ncell]) return;
        int lo = 0, hi = ncell;  // largest cell with t_chunk[cell] <= item
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (t_chunk[mid] <= item) lo = mid; else hi = mid;
        }
        const int cell = lo;
        const int i = t_start[cell] + 32 * (item - t_chunk[cell]) + lane;
        const bool valid = i < t_start[cell + 1];
        const double xi = valid ? txs[i] : 1e150, yi = valid ? tys[i] : 1e150, zi = valid ? tzs[i] : 1e150;
        double a_psi = 0.0, a_x = 0.0, a_y = 0.0, a_z = 0.0;
        int stage_id = 0;
        {
            const int cx = cell % g.nc[0], cy = (cell / g.nc[0]) % g.nc[1], cz = cell / (g.nc[0] * g.nc[1]);
            for (int oz = -g.range[2]; oz <= g.range[2]; ++oz) {
                int nz = cz + oz;
                const int wz = floor_div(nz, g.nc[2]);
                nz -= wz * g.nc[2];
                const double shz = wz * g.L[2];
                for (int oy = -g.range[1]; oy <= g.range[1]; ++oy) {
                    int ny = cy + oy;
                    const int wy = floor_div(ny, g.nc[1]);
                    ny -= wy * g.nc[1];
                    const double shy = wy * g.L[1];
                    for (int ox = -g.range[0]; ox <= g.range[0]; ++ox) {
                        int nx = cx + ox;
                        const int wx = floor_div(nx, g.nc[0]);
                        nx -= wx * g.nc[0];
                        const double shx = wx * g.L[0];
                        const int scell = (nz * g.nc[1] + ny) * g.nc[0] + nx;
                        const int jb = s_start[scell], je = s_start[scell + 1];
                        for (int j0 = jb; j0 < je; j0 += RS_STAGE) {
                            if (SPLIT > 1 && (stage_id++ % SPLIT) != warp) continue;
                            const int cnt = min(RS_STAGE, je - j0);
                            __syncwarp();
#pragma unroll
                            for (int h = 0; h < RS_STAGE / 32; ++h) {
                                const int jj = lane + 32 * h;
                                if (jj < cnt) {
                                    const int j = j0 + jj;
                                    sxy[jj] = make_double2(sxs[j] + shx, sys[j] + shy);
                                    szq[jj] = make_double2(szs[j] + shz, sqs[j]);
                                }
                            }
                            __syncwarp();
                            unsigned long long mask = 0ull;
#pragma unroll 4
                            for (int jj = 0; jj < cnt; ++jj) {
                                const double2 pxy = sxy[jj];
                                const double pz = szq[jj].x;
                                const double dx = xi - pxy.x, dy = yi - pxy.y, dz = zi - pz;
                                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                                if (r2 < k.rc2) mask |= 1ull << jj;
                            }
                            while (mask) {
                                const int jj = __ffsll((long long)mask) - 1;
                                mask &= mask - 1ull;
                                const double2 pxy = sxy[jj], pzq = szq[jj];
                                const double dx = xi - pxy.x, dy = yi - pxy.y, dz = zi - pzq.x;
                                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                                if (r2 == 0.0) { a_psi = fma(k.R0, pzq.y, a_psi); continue; }  // eq. 21
                                double R, gk = 0.0;
                                pair_eval<NS>(k, T, r2, FIELD, R, gk, sh_tab);
                                a_psi = fma(R, pzq.y, a_psi);
                                if (FIELD) {
                                    const double f = gk * pzq.y;
                                    a_x = fma(f, dx, a_x); a_y = fma(f, dy, a_y); a_z = fma(f, dz, a_z);
                                }
                            }
                        }
                    }
                }
            }
        }
        if (SPLIT > 1) {
            sh_part[warp][0][lane] = a_psi;
            if (FIELD) { sh_part[warp][1][lane] = a_x; sh_part[warp][2][lane] = a_y; sh_part[warp][3][lane] = a_z; }
            __syncthreads();
            if (warp != 0) continue;
            a_psi = sh_part[0][0][lane];
            if (FIELD) { a_x = sh_part[0][1][lane]; a_y = sh_part[0][2][lane]; a_z = sh_part[0][3][lane]; }
#pragma unroll
            for (int w = 1; w < SPLIT; ++w) {
                a_psi += sh_part[w][0][lane];
                if (FIELD) { a_x += sh_part[w][1][lane]; a_y += sh_part[w][2][lane]; a_z += sh_part[w][3][lane]; }
            }
        }
        if (valid) {
            psi[i] = a_psi * k.inv_eps;
            if (FIELD) { ex[i] = a_x * k.inv_eps; ey[i] = a_y * k.inv_eps; ez[i] = a_z * k.inv_eps; }
        }
    }
}

// potentials (and fields) at the particles of tb from the charges sb.qs of the particles of sb (same cell geometry)
int real_direct(pce_ctx* c, const Bins& tb, const Bins& sb, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s)
{
    if (tb.n == 0) return PCE_OK;
    PassTimer t(c, PASS_REAL);
    if (sb.n == 0) {
        PCE_CUDA(c, cudaMemsetAsync(psi_s, 0, (size_t)tb.n * sizeof(double), c->st));
        if (field) {
            PCE_CUDA(c, cudaMemsetAsync(ex_s, 0, (size_t)tb.n * sizeof(double), c->st));
            PCE_CUDA(c, cudaMemsetAsync(ey_s, 0, (size_t)tb.n * sizeof(double), c->st));
            PCE_CUDA(c, cudaMemsetAsync(ez_s, 0, (size_t)tb.n * sizeof(double), c->st));
        }
        return PCE_OK;
    }
    PCE_CUDA(c, cudaMemsetAsync(c->work_ctr + 1, 0, sizeof(int), c->st));
    // the table goes to shared memory with a compile-time row stride (192 or 320 intervals); larger tables stay in global memory
    const int ns = c->rt.n_int <= 192 ? 192 : c->rt.n_int <= 320 ? 320 : 0;
    const size_t dyn = (size_t)(field ? RT_STRIDE : RT_DEG + 1) * ns * sizeof(double);
    const int per_sm = ns ? (int)((200 * 1024) / (dyn + 8192 + 1024)) : 8;
    int blocks = c->num_sm * (per_sm < 1 ? 1 : per_sm > 8 ? 8 : per_sm);
    const int need = cdiv(cdiv(tb.n, 32) + tb.ncell, RS_WARPS);  // upper bound of the number of chunks
    if (blocks > need) blocks = need;
    // few chunks (fewer than 4 per SM sub-partition): the CTA shares a chunk, one item per CTA
    const int chunks_ub = cdiv(tb.n, 32) + tb.ncell;
    const bool split = chunks_ub < c->num_sm * 16;
    if (split) blocks = chunks_ub < c->num_sm * 4 ? chunks_ub : c->num_sm * 4;
#define RS_LAUNCH(F, W, S, NS)                                                                                                       \
    do {                                                                                                                             \
        if (dyn > 16 * 1024) PCE_CUDA(c, cudaFuncSetAttribute(k_real_cells<F, W, S, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn)); \
        k_real_cells<F, W, S, NS><<<blocks, W * 32, dyn, c->st>>>(geom_of(tb), c->rk, c->rt, tb.cell_start, tb.chunk_start, tb.xs, tb.ys, tb.zs, \
                                                                  sb.cell_start, sb.xs, sb.ys, sb.zs, sb.qs, psi_s, F ? ex_s : nullptr,      \
                                                                  F ? ey_s : nullptr, F ? ez_s : nullptr, c->work_ctr + 1);                  \
    } while (0)
#define RS_LAUNCH_NS(F, W, S)                                                  \
    do {                                                                       \
        if (ns == 192) RS_LAUNCH(F, W, S, 192);                                \
        else if (ns == 320) RS_LAUNCH(F, W, S, 320);                           \
        else RS_LAUNCH(F, W, S, 0);                                            \
    } while (0)
    if (field) { if (split) RS_LAUNCH_NS(true, RS_SPLIT_WARPS, RS_SPLIT_WARPS); else RS_LAUNCH_NS(true, RS_WARPS, 1); }
    else { if (split) RS_LAUNCH_NS(false, RS_SPLIT_WARPS, RS_SPLIT_WARPS); else RS_LAUNCH_NS(false, RS_WARPS, 1); }
#undef RS_LAUNCH_NS
#undef RS_LAUNCH
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// ---------------------------------------------------------------- cached near field (CSR)
// ---- thread-per-row variants (few candidates per neighbour cell: a warp per row would idle most lanes)
struct OpCount {
    int cnt = 0;
    __device__ __forceinline__ void operator()(int, double, double, double, double) { ++cnt; }
};

__global__ void __launch_bounds__(128)
k_csr_count(int n, CellGeom g, double rc2, const int* __restrict__ cell_start, const double* __restrict__ xs,
            const double* __restrict__ ys, const double* __restrict__ zs, int* __restrict__ row_ptr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    OpCount op;
    for_neighbors(g, cell_start, xs, ys, zs, i, rc2, op);
    row_ptr[i] = op.cnt + 1;  // + the diagonal (self term)
}

struct OpFill {
    const RealConst& k;
    const RealTable& T;
    int* __restrict__ col;
    double* __restrict__ val;
    long long pos;
    __device__ OpFill(const RealConst& k_, const RealTable& T_, int* c_, double* v_, long long p_) : k(k_), T(T_), col(c_), val(v_), pos(p_) {}
    __device__ __forceinline__ void operator()(int j, double, double, double, double r2)
    {
        double R = k.R0, gk;
        if (r2 > 0.0) pair_eval(k, T, r2, false, R, gk);
        col[pos] = j;
        val[pos] = R * k.inv_eps;
        ++pos;
    }
};

__global__ void __launch_bounds__(128)
k_csr_fill(int n, CellGeom g, RealConst k, RealTable T, const int* __restrict__ cell_start, const double* __restrict__ xs,
           const double* __restrict__ ys, const double* __restrict__ zs, const int* __restrict__ row_ptr,
           int* __restrict__ col, double* __restrict__ val, int tab_in_smem)
{
    extern __shared__ double sh_tab[];
    if (tab_in_smem) {
        const int nt = (RT_DEG + 1) * T.n_int;
        for (int e = threadIdx.x; e < nt; e += blockDim.x) sh_tab[e] = T.tab[e];
        __syncthreads();
        T.tab = sh_tab;
    }
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    long long pos = row_ptr[i];
    col[pos] = i;
    val[pos] = k.R0 * k.inv_eps;  // self term, eq. 21
    OpFill op(k, T, col, val, pos + 1);
    for_neighbors(g, cell_start, xs, ys, zs, i, k.rc2, op);
}

// ---- warp-per-row variants (crowded cells)
// One warp per row (sorted bead i): the lanes test the candidates of the 27 neighbour cells 32 at a time; hits are counted
// (k_csr_count) or ranked by ballot, evaluated one per lane and written in candidate order (k_csr_fill): every lane of the
// warp evaluates a kernel, the row's entries are written with coalesced stores, and the order is fixed (deterministic SpMV).
template <bool FILL>
__global__ void __launch_bounds__(256)
k_csr_rows(int n, CellGeom g, RealConst k, RealTable T, const int* __restrict__ cell_start, const double* __restrict__ xs,
           const double* __restrict__ ys, const double* __restrict__ zs, int* __restrict__ row_ptr, int* __restrict__ col,
           double* __restrict__ val, int tab_in_smem)
{
    extern __shared__ double sh_tab[];
    if (FILL && tab_in_smem) {
        const int nt = (RT_DEG + 1) * T.n_int;
        for (int e = threadIdx.x; e < nt; e += blockDim.x) sh_tab[e] = T.tab[e];
        __syncthreads();
        T.tab = sh_tab;
    }
    const int lane = threadIdx.x & 31;
    const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (i >= n) return;
    const double xi = xs[i], yi = ys[i], zi = zs[i];
    const int cx = min((int)(xi * g.inv_cell[0]), g.nc[0] - 1);
    const int cy = min((int)(yi * g.inv_cell[1]), g.nc[1] - 1);
    const int cz = min((int)(zi * g.inv_cell[2]), g.nc[2] - 1);
    long long pos = 0;
    int cnt = 1;  // the diagonal (self term, eq. 21) comes first
    if (FILL) {
        pos = row_ptr[i];
        if (lane == 0) { col[pos] = i; val[pos] = k.R0 * k.inv_eps; }
        ++pos;
    }
    for (int oz = -g.range[2]; oz <= g.range[2]; ++oz) {
        int nz = cz + oz;
        const int wz = floor_div(nz, g.nc[2]);
        nz -= wz * g.nc[2];
        const double sz = wz * g.L[2];
        for (int oy = -g.range[1]; oy <= g.range[1]; ++oy) {
            int ny = cy + oy;
            const int wy = floor_div(ny, g.nc[1]);
            ny -= wy * g.nc[1];
            const double sy = wy * g.L[1];
            for (int ox = -g.range[0]; ox <= g.range[0]; ++ox) {
                int nx = cx + ox;
                const int wx = floor_div(nx, g.nc[0]);
                nx -= wx * g.nc[0];
                const double sx = wx * g.L[0];
                const int cell = (nz * g.nc[1] + ny) * g.nc[0] + nx;
                const int jb = cell_start[cell], je = cell_start[cell + 1];
                const bool home = (ox == 0 && oy == 0 && oz == 0);
                for (int j0 = jb; j0 < je; j0 += 32) {
                    const int j = j0 + lane;
                    bool hit = false;
                    double r2 = 0.0;
                    if (j < je && !(home && j == i)) {
                        const double dx = xi - (xs[j] + sx), dy = yi - (ys[j] + sy), dz = zi - (zs[j] + sz);
                        r2 = dx * dx + dy * dy + dz * dz;
                        hit = r2 < k.rc2;
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, hit);
                    if (FILL) {
                        if (hit) {
                            double R = k.R0, gk;
                            if (r2 > 0.0) pair_eval(k, T, r2, false, R, gk);
                            const long long w = pos + __popc(m & ((1u << lane) - 1u));
                            col[w] = j;
                            val[w] = R * k.inv_eps;
                        }
                        pos += __popc(m);
                    } else {
                        cnt += __popc(m);
                    }
                }
            }
        }
    }
    if (!FILL && lane == 0) row_ptr[i] = cnt;
}

// 64-bit total of the row counts (the int32 scan below would wrap silently past 2^31 entries)
__global__ void __launch_bounds__(256) k_count_total(int n, const int* __restrict__ cnt, unsigned long long* __restrict__ total)
{
    unsigned long long v = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) v += (unsigned)cnt[i];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(total, v);
}

int real_csr_build(pce_ctx* c, const Bins& b)
{
    c->nnz = 0;
    if (b.n == 0) return PCE_OK;
    PassTimer t(c, PASS_REAL);
    const int n = b.n;
    PCE_CUDA(c, cudaMemsetAsync(c->csr_ptr + n, 0, sizeof(int), c->st));
    // crowded cells (>= 32 particles per cell on average, e.g. one 2562-bead sphere inside a few r_c-sized cells) or few rows:
    // one warp per row; otherwise one thread per row
    const bool warp_rows = (double)n / b.ncell >= 32.0 || n < 32768;
    if (warp_rows)
        k_csr_rows<false><<<cdiv((long long)n * 32, 256), 256, 0, c->st>>>(n, geom_of(b), c->rk, c->rt, b.cell_start, b.xs, b.ys, b.zs,
                                                                            c->csr_ptr, nullptr, nullptr, 0);
    else
        k_csr_count<<<cdiv(n, 128), 128, 0, c->st>>>(n, geom_of(b), c->rk.rc2, b.cell_start, b.xs, b.ys, b.zs, c->csr_ptr);
    c->launches++;
    unsigned long long* total_d = reinterpret_cast<unsigned long long*>(c->scal + 32);
    PCE_CUDA(c, cudaMemsetAsync(total_d, 0, sizeof(unsigned long long), c->st));
    k_count_total<<<256, 256, 0, c->st>>>(n, c->csr_ptr, total_d);
    c->launches++;
    int rc = exclusive_scan(c, c->csr_ptr, n + 1);
    if (rc) return rc;
    int nnz = 0;
    unsigned long long total = 0;
    PCE_CUDA(c, cudaMemcpyAsync(&nnz, c->csr_ptr + n, sizeof(int), cudaMemcpyDeviceToHost, c->st));
    PCE_CUDA(c, cudaMemcpyAsync(&total, total_d, sizeof(total), cudaMemcpyDeviceToHost, c->st));
    PCE_CUDA(c, cudaStreamSynchronize(c->st));
    if (total > 0x7fffffffull || nnz < 0 || (unsigned long long)nnz != total) {
        c->err = "near-field entry count overflows int32 (" + std::to_string(total) + " pairs within r_c)";
        return PCE_ENOMEM;
    }
    if (nnz > c->nnz_cap) {
        cudaFree(c->csr_col); cudaFree(c->csr_val);
        c->csr_col = nullptr; c->csr_val = nullptr;
        c->bytes -= c->nnz_cap * 12;
        c->nnz_cap = (long long)(nnz * 1.1) + 1024;
        if (cudaMalloc(&c->csr_col, c->nnz_cap * sizeof(int)) != cudaSuccess ||
            cudaMalloc(&c->csr_val, c->nnz_cap * sizeof(double)) != cudaSuccess) {
            c->err = "out of device memory for the cached near field";
            c->nnz_cap = 0;
            return PCE_ENOMEM;
        }
        c->bytes += c->nnz_cap * 12;
    }
    c->nnz = nnz;
    const size_t tab_bytes = (size_t)(RT_DEG + 1) * c->rt.n_int * sizeof(double);
    const int in_smem = tab_bytes <= 96 * 1024 ? 1 : 0;
    if (warp_rows) {
        if (in_smem && tab_bytes > 40 * 1024) PCE_CUDA(c, cudaFuncSetAttribute(k_csr_rows<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tab_bytes));
        k_csr_rows<true><<<cdiv((long long)n * 32, 256), 256, in_smem ? tab_bytes : 0, c->st>>>(n, geom_of(b), c->rk, c->rt, b.cell_start, b.xs,
                                                                                                 b.ys, b.zs, c->csr_ptr, c->csr_col, c->csr_val, in_smem);
    } else {
        if (in_smem && tab_bytes > 40 * 1024) PCE_CUDA(c, cudaFuncSetAttribute(k_csr_fill, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tab_bytes));
        k_csr_fill<<<cdiv(n, 128), 128, in_smem ? tab_bytes : 0, c->st>>>(n, geom_of(b), c->rk, c->rt, b.cell_start, b.xs, b.ys, b.zs, c->csr_ptr,
                                                                          c->csr_col, c->csr_val, in_smem);
    }
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// one warp per row; x = b.qs (sorted charges), y = psi_s (sorted)
__global__ void __launch_bounds__(256)
k_csr_spmv(int n, const int* __restrict__ row_ptr, const int* __restrict__ col, const double* __restrict__ val,
           const double* __restrict__ x, double* __restrict__ y, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    const int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (row >= n) return;
    const int b = row_ptr[row], e = row_ptr[row + 1];
    double s = 0.0;
    for (int k = b + lane; k < e; k += 32) s += val[k] * x[col[k]];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if (lane == 0) y[row] = s;
}

int real_csr_spmv(pce_ctx* c, const Bins& b, double* psi_s)
{
    if (b.n == 0) return PCE_OK;
    PassTimer t(c, PASS_REAL);
    k_csr_spmv<<<cdiv((long long)b.n * 32, 256), 256, 0, c->st>>>(b.n, c->csr_ptr, c->csr_col, c->csr_val, b.qs, psi_s, c->skip_flag);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
