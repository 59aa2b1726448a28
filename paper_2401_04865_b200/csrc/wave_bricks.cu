// wave_bricks.cu -- output-stationary Gaussian spreading (eq. 25) and
// brick-stationary Gaussian gather (eq. 27) for sm_100a.
//
// The paper spreads with one block of P^3 threads per particle and global atomics
// (PAPER.md:263).  Here the mesh is cut into 8^3 bricks and ONE WARP owns one brick: lane l
// holds, for all 8 planes, the points (y = l/4, x = 2(l%4), 2(l%4)+1) in 16 fp64 REGISTERS
// (the mma D / B fragment layout).  Warps never synchronise with each other (one
// __syncthreads after the table load, none afterwards):
//   1. particles are binned by 8-point mesh bin (counting sort, cells.cu; bins shifted by
//      P/2 mod 8 so that the cells whose support meets a brick span ceil((P+7)/8) bins per
//      dimension); the warp enumerates the contiguous runs of the sorted particle list in
//      those bins and walks them as one flat candidate list;
//   2. test: one candidate per lane (one 16-byte load: the first support index per
//      dimension), ballot, hits appended to a per-warp queue in shared memory;
//   3. every 32 hits: lane l computes the 3x8 brick-local window weights of hit l.  With
//      u = u0 + r the offset of support point r from the particle (mesh units),
//          W(r) = exp(-aw u^2),  W(r+1) = W(r) t(r),  t(r+1) = t(r) exp(-2 aw),
//      started from per-particle coefficients of k_window_coef (phi = -s0 mod 8,
//      e1 = exp(-2 aw u0), c0 = exp(-aw u0^2) e1^phi, e8 = e1^8):
//      W(phi + 8m) = c0 e8^m exp(-aw (phi + 8m)^2), t(r) = e1 exp(-aw (2r + 1)); no exp here;
//   4. accumulate on the fp64 tensor path (mma.sync m8n8k4.f64, measured 37.1 TFLOP/s against 33.3 for DFMA chains):
//      per brick the spread is the contraction H_z[y][x] = sum_h (wy_h[y] q_h wz_h[z]) wx_h[x] over the hits h of
//      the brick, the gather T_z[h][x] = sum_y wy_h[y] H~_z[y][x]; see the kernels.
// Spread writes every mesh point exactly once (no atomics, no memset, deterministic).
// Gather keeps the brick of H~ in registers as the mma B operand, handles 8 hits per step and
// issues one global fp64 atomicAdd per hit and quantity.  The window is the truncated Gaussian of eq. 25 on exactly the P^3
// nearest mesh points (reading A5), identical in both passes, so the mesh operator stays
// symmetric.  Grids with Ng % 8 != 0 or Ng - P < 8 take a generic weight routine (direct
// exp, wrap-aware); everything else is shared.
#include "pce_internal.h"

constexpr int BR = 8;          // brick edge in mesh points
constexpr int BWARPS = 4;      // warps (bricks) per CTA
constexpr int MAXPIECE = 96;   // runs of candidates per brick: <= 6 x 6 rows x 2 wrap pieces (P <= 32)
constexpr int STRIDE_PSI = 26; // doubles per hit in the weight table: 3 x 8 + 2 pad (13 x 16 B: conflict-free rows)
constexpr int STRIDE_FLD = 50; // with the field: 3 x (8 w + 8 w u) + 2 pad (25 x 16 B)
constexpr int NTAB = 48 + 48;  // Gt[r + 8] = exp(-aw r^2), Ht[r + 8] = exp(-aw (2r + 1)), r = -8..39

struct WinCoefPtrs {
    const int4* s0;       // [n]
    const double4* cf;    // [3 n]: (c0, e1, e8, 1/e8) of particle p, dimension d at 3 p + d
};

template <int STRIDE>
struct alignas(16) WarpSmem {
    double wt[32 * STRIDE];
    int qidx[64];
    int p_start[MAXPIECE];
    int p_prefix[MAXPIECE + 4];
};

__device__ __forceinline__ int wrap_once(int d, int n) { if (d < 0) d += n; if (d >= n) d -= n; return d; }

// bins (of BR shifted mesh cells) that can hold a particle whose support meets [b0, b0 + bw): the particle's
// mesh cell i0 = floor(x/h) lies in [b0 - P/2, b0 + bw + P/2 - 2] (mod ng); bins are over (i0 + shift) mod ng.
__device__ __forceinline__ int dim_bin_ranges(int b0, int bw, int P, int ng, int nc, int lo[2], int hi[2])
{
    const int shift = (P / 2) % BR;
    const int a = b0 - P / 2 + shift, b = b0 + bw + P / 2 - 2 + shift;
    if (b - a + 1 >= ng) { lo[0] = 0; hi[0] = nc - 1; return 1; }
    const int aw = wrap_once(wrap_once(a, ng), ng), bwp = wrap_once(wrap_once(b, ng), ng);
    if (aw <= bwp) { lo[0] = aw / BR; hi[0] = bwp / BR; return 1; }
    if (bwp / BR >= aw / BR) { lo[0] = 0; hi[0] = nc - 1; return 1; }
    lo[0] = 0; hi[0] = bwp / BR; lo[1] = aw / BR; hi[1] = nc - 1;
    return 2;
}

struct Brick {
    int b0[3], bw[3];
    int npiece, M;
};

// brick of this warp and its candidate runs (p_start / p_prefix in the warp's shared memory)
template <int STRIDE>
__device__ __forceinline__ bool brick_setup(const WaveConst& wc, int nbx, int nby, int nbz, const int* __restrict__ cell_start,
                                            WarpSmem<STRIDE>& s, Brick& br, int lane, int brick_id)
{
    if (brick_id >= nbx * nby * nbz) return false;
    int t = brick_id;
    const int bx = t % nbx; t /= nbx;
    const int by = t % nby, bz = t / nby;
    br.b0[0] = bx * BR; br.b0[1] = by * BR; br.b0[2] = bz * BR;
    br.bw[0] = min(BR, wc.Ng[0] - br.b0[0]); br.bw[1] = min(BR, wc.Ng[1] - br.b0[1]); br.bw[2] = min(BR, wc.Ng[2] - br.b0[2]);
    int lox[2], hix[2], loy[2], hiy[2], loz[2], hiz[2];
    const int nrx = dim_bin_ranges(br.b0[0], br.bw[0], wc.P, wc.Ng[0], nbx, lox, hix);
    const int nry = dim_bin_ranges(br.b0[1], br.bw[1], wc.P, wc.Ng[1], nby, loy, hiy);
    const int nrz = dim_bin_ranges(br.b0[2], br.bw[2], wc.P, wc.Ng[2], nbz, loz, hiz);
    const int n0y = hiy[0] - loy[0] + 1, n0z = hiz[0] - loz[0] + 1;
    const int cnty = n0y + (nry == 2 ? hiy[1] - loy[1] + 1 : 0);  // bins in y
    const int cntz = n0z + (nrz == 2 ? hiz[1] - loz[1] + 1 : 0);  // bins in z
    // pieces: (z bin, y bin, x run)
    const int npiece = cntz * cnty * nrx;
    br.npiece = npiece;  // <= MAXPIECE by construction (P <= 32)
    int carry = 0;
    for (int base = 0; base < npiece; base += 32) {
        const int k = base + lane;
        int len = 0, start = 0;
        if (k < npiece) {
            const int xr = (nrx == 2) ? (k & 1) : 0;
            const int r = (nrx == 2) ? (k >> 1) : k;
            const int zi = r / cnty, yi = r - zi * cnty;
            const int yb = (yi < n0y) ? loy[0] + yi : loy[1] + (yi - n0y);
            const int zb = (zi < n0z) ? loz[0] + zi : loz[1] + (zi - n0z);
            const int row = (zb * nby + yb) * nbx;
            start = cell_start[row + (xr ? lox[1] : lox[0])];
            len = cell_start[row + (xr ? hix[1] : hix[0]) + 1] - start;
        }
        int incl = len;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += v;
        }
        if (k < npiece) { s.p_start[k] = start; s.p_prefix[k] = carry + incl - len; }
        carry += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) s.p_prefix[npiece] = carry;
    br.M = carry;
    __syncwarp();
    return true;
}

__device__ __forceinline__ bool support_meets_brick(const WaveConst& wc, const Brick& br, const int4 s0)
{
    const int sv[3] = {s0.x, s0.y, s0.z};
    bool hit = true;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int ng = wc.Ng[d];
        const int dsl = wrap_once(br.b0[d] - sv[d], ng);  // brick origin - first support index, mod ng
        hit = hit && (dsl < wc.P || dsl + br.bw[d] > ng);
    }
    return hit;
}

// the 8 brick-local window weights of one particle in one dimension (0 outside the support), and with FIELD the
// weights times u = (mesh index - x/h).  tab = [Gt | Ht] in shared memory.
//   fast path (ng % 8 == 0, ng - P >= 8): the support meets the brick in one run, brick-local j <-> r = r0 + j
//   generic path: direct exp per point, periodic wrap per point
template <bool FIELD>
__device__ __forceinline__ void brick_weights(const WaveConst& wc, const double* __restrict__ tab, bool generic, int b0, int ng,
                                              int s0, const double4 cf, double u0, double scale, double* __restrict__ w)
{
    const int P = wc.P;
    const int dsl = wrap_once(b0 - s0, ng);
    double v[BR], vu[BR];
    if (!generic) {
        const int r0 = (dsl < P) ? dsl : dsl - ng;
        const int phi = (-s0) & (BR - 1);
        const int m = (r0 - phi) >> 3;  // -1 .. 3
        const double e82 = cf.z * cf.z;
        const double pm = (m < 0) ? cf.w : (m == 0) ? 1.0 : (m == 1) ? cf.z : (m == 2) ? e82 : e82 * cf.z;
        double pw = cf.x * pm * tab[r0 + 8] * scale;
        double t = cf.y * tab[48 + r0 + 8];
        const double g2 = tab[9] * tab[9];  // exp(-2 aw)
#pragma unroll
        for (int j = 0; j < BR; ++j) {
            const int r = r0 + j;
            v[j] = ((unsigned)r < (unsigned)P) ? pw : 0.0;
            if (FIELD) vu[j] = v[j] * (u0 + (double)r);
            pw *= t;
            t *= g2;
        }
    } else {
        int r = dsl;
#pragma unroll
        for (int j = 0; j < BR; ++j) {
            const double u = u0 + (double)r;
            v[j] = (r < P) ? scale * exp(-wc.aw * u * u) : 0.0;
            if (FIELD) vu[j] = v[j] * u;
            if (++r == ng) r = 0;
        }
    }
#pragma unroll
    for (int j = 0; j < BR; j += 2) *reinterpret_cast<double2*>(w + j) = make_double2(v[j], v[j + 1]);
    if (FIELD) {
#pragma unroll
        for (int j = 0; j < BR; j += 2) *reinterpret_cast<double2*>(w + BR + j) = make_double2(vu[j], vu[j + 1]);
    }
}

__device__ __forceinline__ void load_tables(const WaveConst& wc, double* tab)
{
    for (int k = threadIdx.x; k < NTAB; k += blockDim.x) {
        const int r = (k < 48 ? k : k - 48) - 8;
        tab[k] = (k < 48) ? exp(-wc.aw * (double)(r * r)) : exp(-wc.aw * (double)(2 * r + 1));
    }
    __syncthreads();
}

// hits appended by the test phase; PROCESS consumes the first min(nq, 32).  Each lane walks the runs forwards:
// its candidates c = lane, lane + 32, ... only ever move to later runs.
#define BRICK_WALK(PROCESS)                                                                        \
    int nq = 0, pc = 0;                                                                            \
    for (int cb = 0; cb < br.M; cb += 32) {                                                        \
        const int c = cb + lane;                                                                   \
        bool hit = false;                                                                          \
        int pi = 0;                                                                                \
        if (c < br.M) {                                                                            \
            while (c >= s.p_prefix[pc + 1]) ++pc;                                                  \
            pi = s.p_start[pc] + (c - s.p_prefix[pc]);                                             \
            hit = support_meets_brick(wc, br, wp.s0[pi]);                                          \
        }                                                                                          \
        const unsigned m = __ballot_sync(0xffffffffu, hit);                                        \
        if (hit) s.qidx[nq + __popc(m & ((1u << lane) - 1u))] = pi;                                \
        nq += __popc(m);                                                                           \
        __syncwarp();                                                                              \
        if (nq >= 32) {                                                                            \
            PROCESS(32);                                                                           \
            const int rest = nq - 32;                                                              \
            const int v = (lane < rest) ? s.qidx[32 + lane] : 0;                                   \
            __syncwarp();                                                                          \
            if (lane < rest) s.qidx[lane] = v;                                                     \
            nq = rest;                                                                             \
            __syncwarp();                                                                          \
        }                                                                                          \
    }                                                                                              \
    if (nq > 0) { PROCESS(nq); }

// ---------------------------------------------------------------- window coefficients (once per position update)
__global__ void __launch_bounds__(256)
k_window_coef(int n, WaveConst wc, const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
              int4* __restrict__ s0o, double4* __restrict__ cfo)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double pos[3] = {xs[i], ys[i], zs[i]};
    int sv[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double xd = pos[d] * wc.inv_h[d];
        const int i0 = min((int)xd, wc.Ng[d] - 1);
        const int s0 = i0 - wc.P / 2 + 1;  // first support index (reading A5, even P); may be negative
        const double u0 = (double)s0 - xd; // in (-P/2, -P/2 + 1]
        const int phi = (-s0) & (BR - 1);
        sv[d] = s0;
        cfo[3 * (size_t)i + d] = make_double4(exp(-wc.aw * u0 * (u0 + 2.0 * phi)), exp(-2.0 * wc.aw * u0), exp(-16.0 * wc.aw * u0),
                                              exp(16.0 * wc.aw * u0));
    }
    s0o[i] = make_int4(sv[0], sv[1], sv[2], 0);
}

// weights of the first nh queued hits, one hit per lane, into the warp's table
#define BRICK_WEIGHTS(FIELD_, STRIDE_, DW_, QSCALE)                                                                     \
    if (lane < nh) {                                                                                                    \
        const int p = s.qidx[lane];                                                                                     \
        double* w = s.wt + lane * (STRIDE_);                                                                            \
        const int4 s0v = wp.s0[p];                                                                                      \
        const int sv[3] = {s0v.x, s0v.y, s0v.z};                                                                        \
        double u0[3] = {0.0, 0.0, 0.0};                                                                                 \
        if ((FIELD_) || generic) {                                                                                      \
            u0[0] = (double)sv[0] - xs[p] * wc.inv_h[0];                                                                \
            u0[1] = (double)sv[1] - ys[p] * wc.inv_h[1];                                                                \
            u0[2] = (double)sv[2] - zs[p] * wc.inv_h[2];                                                                \
        }                                                                                                               \
        const double qscale = (QSCALE);                                                                                 \
        _Pragma("unroll") for (int d = 0; d < 3; ++d)                                                                   \
            brick_weights<FIELD_>(wc, tab, generic, br.b0[d], wc.Ng[d], sv[d], wp.cf[3 * (size_t)p + d], u0[d],         \
                                  d == 2 ? qscale : 1.0, w + (DW_) * d);                                                \
    }                                                                                                                   \
    __syncwarp();

// ---------------------------------------------------------------- fp64 tensor-core step
// D(8x8) += A(8x4) B(4x8), fp64 (mma.sync m8n8k4; tcgen05 has no fp64 kind).  With g = lane/4, t = lane%4 a lane holds
// A[g][t], B[t][g] and the pair D[g][2t], D[g][2t+1].
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// ---------------------------------------------------------------- spread
// Per brick and mesh plane z the spread is a dense contraction over the hits h of the brick:
//     H_z[y][x] = sum_h (wy_h[y] q_h wz_h[z]) wx_h[x]  =  (A_z B)[y][x],  A_z = 8 x hits, B = hits x 8,
// issued four hits at a time as one fp64 mma per plane: 8 DMUL + 8 DMMA per 4 hits instead of 16 DMUL + 64 DFMA.
__global__ void __launch_bounds__(BWARPS * 32, 6)
k_spread_bricks(WaveConst wc, int nbx, int nby, int nbz, const int* __restrict__ cell_start, WinCoefPtrs wp,
                const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                const double* __restrict__ qs, double* __restrict__ grid, int vec_ok, int generic_, int* __restrict__ work_ctr,
                const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* tab = reinterpret_cast<double*>(smem_raw);
    WarpSmem<STRIDE_PSI>* sm = reinterpret_cast<WarpSmem<STRIDE_PSI>*>(smem_raw + NTAB * sizeof(double));
    load_tables(wc, tab);
    const bool generic = generic_ != 0;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem<STRIDE_PSI>& s = sm[warp];
    const int g = lane >> 2, t = lane & 3;  // mma fragment coordinates
    for (;;) {  // persistent warps: bricks are handed out by a global counter
    int brick_id = 0;
    if (lane == 0) brick_id = atomicAdd(work_ctr, 1);
    brick_id = __shfl_sync(0xffffffffu, brick_id, 0);
    Brick br;
    if (!brick_setup(wc, nbx, nby, nbz, cell_start, s, br, lane, brick_id)) return;
    double acc[BR][2];  // plane z: H[z][y = g][x = 2t, 2t + 1]
#pragma unroll
    for (int z = 0; z < BR; ++z) { acc[z][0] = 0.0; acc[z][1] = 0.0; }

#define SPREAD_PROCESS(NH)                                                                                              \
    {                                                                                                                   \
        const int nh = (NH);                                                                                            \
        BRICK_WEIGHTS(false, STRIDE_PSI, BR, qs[p])                                                                     \
        for (int sb = 0; sb < nh; sb += 4) {                                                                            \
            const bool live = sb + t < nh;                           /* rows >= nh were never written: read row 0 */   \
            const double* w = s.wt + (live ? sb + t : 0) * STRIDE_PSI;                                                  \
            const double bx = live ? w[g] : 0.0;                      /* B[t][g] = wx_h[x = g]            */            \
            const double ay = live ? w[BR + g] : 0.0;                 /* wy_h[y = g]                      */            \
            double wz[BR];                                            /* q_h wz_h[0..7]                   */            \
            _Pragma("unroll") for (int z = 0; z < BR; z += 2) {                                                         \
                const double2 v = *reinterpret_cast<const double2*>(w + 2 * BR + z);                                    \
                wz[z] = v.x; wz[z + 1] = v.y;                                                                           \
            }                                                                                                           \
            _Pragma("unroll") for (int z = 0; z < BR; ++z) dmma884(acc[z][0], acc[z][1], ay * wz[z], bx);               \
        }                                                                                                               \
        __syncwarp();                                                                                                   \
    }

    BRICK_WALK(SPREAD_PROCESS)
#undef SPREAD_PROCESS

    const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
    const int gx = br.b0[0] + 2 * t, gy = br.b0[1] + g;
    if (gy < wc.Ng[1]) {
#pragma unroll
        for (int z = 0; z < BR; ++z) {
            const int gz = br.b0[2] + z;
            if (gz >= wc.Ng[2]) break;
            double* row = grid + ((size_t)gz * Ny + gy) * Nx + gx;
            if (vec_ok && gx + 1 < wc.Ng[0]) {
                *reinterpret_cast<double2*>(row) = make_double2(acc[z][0], acc[z][1]);
            } else {
                if (gx < wc.Ng[0]) row[0] = acc[z][0];
                if (gx + 1 < wc.Ng[0]) row[1] = acc[z][1];
            }
        }
    }
    __syncwarp();
    }  // next brick
}
// ---------------------------------------------------------------- gather
// Per brick, plane z and group of 8 hits the gather is the contraction  T_z[h][x] = sum_y wy_h[y] H~_z[y][x]  (two fp64
// mma k-steps, the brick of H~ being the B operand held in registers), followed by  U[h][x] += wz_h[z] T_z[h][x]  and, after
// the 8 planes,  psi_h += sum_x wx_h[x] U[h][x]  (4-lane shuffle, one atomicAdd per hit and quantity).  With the field the
// window-gradient sums (reading A3) reuse T_z with wz u_z and wx u_x, and need a second contraction with wy u_y.
template <bool FIELD>
__global__ void __launch_bounds__(BWARPS * 32, FIELD ? 3 : 6)
k_gather_bricks(WaveConst wc, int nbx, int nby, int nbz, const int* __restrict__ cell_start, WinCoefPtrs wp,
                const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                const double* __restrict__ grid, double* __restrict__ psi, double* __restrict__ ex, double* __restrict__ ey,
                double* __restrict__ ez, int vec_ok, int generic_, int* __restrict__ work_ctr, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    constexpr int STRIDE = FIELD ? STRIDE_FLD : STRIDE_PSI;
    constexpr int DW = FIELD ? 2 * BR : BR;  // doubles per dimension in the weight table
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* tab = reinterpret_cast<double*>(smem_raw);
    WarpSmem<STRIDE>* sm = reinterpret_cast<WarpSmem<STRIDE>*>(smem_raw + NTAB * sizeof(double));
    load_tables(wc, tab);
    const bool generic = generic_ != 0;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem<STRIDE>& s = sm[warp];
    const int g = lane >> 2, t = lane & 3;  // mma fragment coordinates
    (void)vec_ok;
    for (;;) {  // persistent warps: bricks are handed out by a global counter
    int brick_id = 0;
    if (lane == 0) brick_id = atomicAdd(work_ctr, 1);
    brick_id = __shfl_sync(0xffffffffu, brick_id, 0);
    Brick br;
    if (!brick_setup(wc, nbx, nby, nbz, cell_start, s, br, lane, brick_id)) return;
    if (br.M == 0) continue;
    // B operands: H[z][0] = H~[z][y = t][x = g], H[z][1] = H~[z][y = t + 4][x = g]  (0 outside the mesh)
    double H[BR][2];
    {
        const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
        const int gx = br.b0[0] + g;
#pragma unroll
        for (int z = 0; z < BR; ++z) {
            const int gz = br.b0[2] + z;
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int gy = br.b0[1] + t + 4 * k;
                const bool ok = gz < wc.Ng[2] && gy < wc.Ng[1] && gx < wc.Ng[0];
                H[z][k] = ok ? grid[((size_t)gz * Ny + gy) * Nx + gx] : 0.0;
            }
        }
    }

#define GATHER_PROCESS(NH)                                                                                              \
    {                                                                                                                   \
        const int nh = (NH);                                                                                            \
        BRICK_WEIGHTS(FIELD, STRIDE, DW, 1.0)                                                                           \
        for (int sb = 0; sb < nh; sb += 8) {                                                                            \
            const int hr = sb + g;                                                                                      \
            const bool live = hr < nh;                                                                                  \
            const double* w = s.wt + (live ? hr : 0) * STRIDE;                                                          \
            const double a0 = live ? w[DW + t] : 0.0, a1 = live ? w[DW + t + 4] : 0.0;          /* wy_h[y]    */        \
            const double2 wx2 = *reinterpret_cast<const double2*>(w + 2 * t);                   /* wx_h[2t..] */        \
            double wz[BR];                                                                                              \
            _Pragma("unroll") for (int z = 0; z < BR; z += 2) {                                                         \
                const double2 v = *reinterpret_cast<const double2*>(w + 2 * DW + z);                                    \
                wz[z] = v.x; wz[z + 1] = v.y;                                                                           \
            }                                                                                                           \
            if (!FIELD) {                                                                                               \
                double u0 = 0.0, u1 = 0.0;                                                                              \
                _Pragma("unroll") for (int z = 0; z < BR; ++z) {                                                        \
                    double t0 = 0.0, t1 = 0.0;                                                                          \
                    dmma884(t0, t1, a0, H[z][0]);                                                                       \
                    dmma884(t0, t1, a1, H[z][1]);                                                                       \
                    u0 = fma(wz[z], t0, u0); u1 = fma(wz[z], t1, u1);                                                   \
                }                                                                                                       \
                double r = fma(wx2.y, u1, wx2.x * u0);                                                                  \
                r += __shfl_xor_sync(0xffffffffu, r, 1);                                                                \
                r += __shfl_xor_sync(0xffffffffu, r, 2);                                                                \
                if (live && t == 0) atomicAdd(&psi[s.qidx[hr]], r);                                                     \
            } else {                                                                                                    \
                const double b0 = live ? w[DW + BR + t] : 0.0, b1 = live ? w[DW + BR + t + 4] : 0.0;  /* wy u_y */      \
                const double2 wxu2 = *reinterpret_cast<const double2*>(w + BR + 2 * t);               /* wx u_x */      \
                double wzu[BR];                                                                                         \
                _Pragma("unroll") for (int z = 0; z < BR; z += 2) {                                                     \
                    const double2 v = *reinterpret_cast<const double2*>(w + 2 * DW + BR + z);                           \
                    wzu[z] = v.x; wzu[z + 1] = v.y;                                                                     \
                }                                                                                                       \
                double u0 = 0.0, u1 = 0.0, uz0 = 0.0, uz1 = 0.0, uy0 = 0.0, uy1 = 0.0;                                  \
                _Pragma("unroll") for (int z = 0; z < BR; ++z) {                                                        \
                    double t0 = 0.0, t1 = 0.0, v0 = 0.0, v1 = 0.0;                                                      \
                    dmma884(t0, t1, a0, H[z][0]);                                                                       \
                    dmma884(t0, t1, a1, H[z][1]);                                                                       \
                    dmma884(v0, v1, b0, H[z][0]);                                                                       \
                    dmma884(v0, v1, b1, H[z][1]);                                                                       \
                    u0 = fma(wz[z], t0, u0); u1 = fma(wz[z], t1, u1);                                                   \
                    uz0 = fma(wzu[z], t0, uz0); uz1 = fma(wzu[z], t1, uz1);                                             \
                    uy0 = fma(wz[z], v0, uy0); uy1 = fma(wz[z], v1, uy1);                                               \
                }                                                                                                       \
                double r0 = fma(wx2.y, u1, wx2.x * u0);      /* psi                  */                                 \
                double r1 = fma(wxu2.y, u1, wxu2.x * u0);    /* sum W u_x H          */                                 \
                double r2 = fma(wx2.y, uy1, wx2.x * uy0);    /* sum W u_y H          */                                 \
                double r3 = fma(wx2.y, uz1, wx2.x * uz0);    /* sum W u_z H          */                                 \
                r0 += __shfl_xor_sync(0xffffffffu, r0, 1); r1 += __shfl_xor_sync(0xffffffffu, r1, 1);                   \
                r2 += __shfl_xor_sync(0xffffffffu, r2, 1); r3 += __shfl_xor_sync(0xffffffffu, r3, 1);                   \
                r0 += __shfl_xor_sync(0xffffffffu, r0, 2); r1 += __shfl_xor_sync(0xffffffffu, r1, 2);                   \
                r2 += __shfl_xor_sync(0xffffffffu, r2, 2); r3 += __shfl_xor_sync(0xffffffffu, r3, 2);                   \
                if (live) {                                                                                             \
                    const int p = s.qidx[hr];                                                                           \
                    /* E = -grad_a, dW/dx_a = +grad_fac u W; lane t issues quantity t */                                \
                    if (t == 0) atomicAdd(&psi[p], r0);                                                                 \
                    else if (t == 1) atomicAdd(&ex[p], -wc.grad_fac[0] * r1);                                           \
                    else if (t == 2) atomicAdd(&ey[p], -wc.grad_fac[1] * r2);                                           \
                    else atomicAdd(&ez[p], -wc.grad_fac[2] * r3);                                                       \
                }                                                                                                       \
            }                                                                                                           \
        }                                                                                                               \
        __syncwarp();                                                                                                   \
    }

    BRICK_WALK(GATHER_PROCESS)
#undef GATHER_PROCESS
    __syncwarp();
    }  // next brick
}

// ---------------------------------------------------------------- host
static size_t smem_bytes(bool field)
{
    return NTAB * sizeof(double) + BWARPS * (field ? sizeof(WarpSmem<STRIDE_FLD>) : sizeof(WarpSmem<STRIDE_PSI>));
}

int wave_bricks_init(pce_ctx* c)
{
    PCE_CUDA(c, cudaFuncSetAttribute(k_spread_bricks, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(false)));
    PCE_CUDA(c, cudaFuncSetAttribute(k_gather_bricks<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(false)));
    PCE_CUDA(c, cudaFuncSetAttribute(k_gather_bricks<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(true)));
    int dev = 0;
    PCE_CUDA(c, cudaGetDevice(&dev));
    PCE_CUDA(c, cudaDeviceGetAttribute(&c->num_sm, cudaDevAttrMultiProcessorCount, dev));
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_spread, k_spread_bricks, BWARPS * 32, smem_bytes(false)));
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_gather, k_gather_bricks<false>, BWARPS * 32, smem_bytes(false)));
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_gather_f, k_gather_bricks<true>, BWARPS * 32, smem_bytes(true)));
    if (c->occ_spread < 1 || c->occ_gather < 1 || c->occ_gather_f < 1) { c->err = "brick kernels do not fit on this device"; return PCE_ECUDA; }
    PCE_CUDA(c, cudaMalloc(&c->work_ctr, 4 * sizeof(int)));
    return PCE_OK;
}

int wave_coef_alloc(pce_ctx* c, Bins& b)
{
    const size_t n = (size_t)(b.n > 0 ? b.n : 1);
    PCE_CUDA(c, cudaMalloc(&b.ws0, n * sizeof(int4)));
    PCE_CUDA(c, cudaMalloc(&b.wcf, 3 * n * sizeof(double4)));
    c->bytes += (long long)(n * 112);
    return PCE_OK;
}

// per-particle window coefficients of a mesh binning (after bins_build)
int wave_window_coef(pce_ctx* c, const Bins& b)
{
    if (b.n == 0) return PCE_OK;
    k_window_coef<<<cdiv(b.n, 256), 256, 0, c->st>>>(b.n, c->wk, b.xs, b.ys, b.zs, b.ws0, b.wcf);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

static WinCoefPtrs coef_ptrs(const Bins& b)
{
    WinCoefPtrs p;
    p.s0 = b.ws0; p.cf = b.wcf;
    return p;
}

// the fast weight routine needs bricks aligned with the periodic mesh and a support that meets a brick in one run
static int generic_weights(const pce_ctx* c)
{
    for (int d = 0; d < 3; ++d)
        if (c->wk.Ng[d] % BR != 0 || c->wk.Ng[d] - c->wk.P < BR) return 1;
    return 0;
}

// persistent grid: as many CTAs as fit on the device (occupancy query at init), never more than there are bricks
static int grid_for(const pce_ctx* c, int per_sm, int nbrick)
{
    const int want = c->num_sm * per_sm, need = cdiv(nbrick, BWARPS);
    return want < need ? want : need;
}

int wave_spread_bricks(pce_ctx* c, const Bins& b)
{
    PassTimer t(c, PASS_SPREAD);
    const int vec_ok = (c->wk.Ng[0] % 2 == 0) ? 1 : 0;
    PCE_CUDA(c, cudaMemsetAsync(c->work_ctr, 0, sizeof(int), c->st));
    k_spread_bricks<<<grid_for(c, c->occ_spread, b.ncell), BWARPS * 32, smem_bytes(false), c->st>>>(c->wk, b.nc[0], b.nc[1], b.nc[2], b.cell_start,
                                                                                     coef_ptrs(b), b.xs, b.ys, b.zs, b.qs, c->grid, vec_ok, generic_weights(c), c->work_ctr, c->skip_flag);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

int wave_gather_bricks(pce_ctx* c, const Bins& b, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s)
{
    if (b.n == 0) return PCE_OK;
    PassTimer t(c, PASS_GATHER);
    const int vec_ok = (c->wk.Ng[0] % 2 == 0) ? 1 : 0;
    const int blocks = grid_for(c, field ? c->occ_gather_f : c->occ_gather, b.ncell);
    PCE_CUDA(c, cudaMemsetAsync(c->work_ctr, 0, sizeof(int), c->st));
    PCE_CUDA(c, cudaMemsetAsync(psi_s, 0, (size_t)b.n * sizeof(double), c->st));
    if (field) {
        PCE_CUDA(c, cudaMemsetAsync(ex_s, 0, (size_t)b.n * sizeof(double), c->st));
        PCE_CUDA(c, cudaMemsetAsync(ey_s, 0, (size_t)b.n * sizeof(double), c->st));
        PCE_CUDA(c, cudaMemsetAsync(ez_s, 0, (size_t)b.n * sizeof(double), c->st));
        k_gather_bricks<true><<<blocks, BWARPS * 32, smem_bytes(true), c->st>>>(c->wk, b.nc[0], b.nc[1], b.nc[2], b.cell_start,
                                                                               coef_ptrs(b), b.xs, b.ys, b.zs, c->grid, psi_s, ex_s, ey_s,
                                                                               ez_s, vec_ok, generic_weights(c), c->work_ctr, c->skip_flag);
    } else {
        k_gather_bricks<false><<<blocks, BWARPS * 32, smem_bytes(false), c->st>>>(c->wk, b.nc[0], b.nc[1], b.nc[2], b.cell_start,
                                                                                 coef_ptrs(b), b.xs, b.ys, b.zs, c->grid, psi_s, nullptr,
                                                                                 nullptr, nullptr, vec_ok, generic_weights(c), c->work_ctr, c->skip_flag);
    }
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
