// wave_tiles.cu -- output-stationary Gaussian spreading (eq. 25) and
// tile-stationary Gaussian gather (eq. 27) for sm_100a.
//
// The paper spreads with one block of P^3 threads per particle and global atomics
// (PAPER.md:263).  Here the mesh is cut into 16^3 tiles, one CTA per tile, 8 warps per CTA,
// one 8^3 brick per warp, one 4x4 (x,y) patch at one z per lane held in 16 fp64 REGISTERS.
// Particles are binned by tile (counting sort); a CTA walks the <= 27 neighbouring bins in
// batches of 128 candidates:
//   phase A  load candidates, test support/tile overlap, ballot-compact (fixed order)
//   phase B  per (particle, dimension): the 16 tile-local window weights from
//            exp(-aw(u0+r)^2) = e0 * e1^r * G[r]  (2 exp + P multiplies instead of 16 exp)
//   phase C  per warp: ballot the particles whose support meets its brick; per hit
//            16 DFMA + 4 DMUL per lane from 5 shared-memory loads
// Spread writes every mesh point exactly once (no atomics, no memset, deterministic).
// Gather keeps the tile of H~ in registers, reduces the 32 lane partials of 8 (or 4x4 with
// field) particles at a time by a transposing butterfly, sums the 8 warps in shared memory
// and issues one global fp64 atomicAdd per particle, tile and quantity.
// The window is the truncated Gaussian of eq. 25 on exactly the P^3 nearest mesh points
// (reading A5), identical in both passes, so the mesh operator stays symmetric.
#include "pce_internal.h"

constexpr int WT = 16;          // tile edge in mesh points
constexpr int WBATCH = 128;     // candidate particles per batch
constexpr int WTHREADS = 256;   // 8 warps = 8 bricks of 8^3
constexpr int MAXR = 32;        // candidate bin ranges per tile (<= 9 rows x 2 wrap pieces)

struct TileSmem {
    double wt[WBATCH][3][WT];   // window weights per accepted particle, dimension, tile-local index (0 outside the support)
    double ub[WBATCH][3];       // u = (mesh index - x/h) at the first support point
    int d[WBATCH][3];           // (tile origin - first support index) mod Ng
    int pidx[WBATCH];           // sorted particle slot
    double q[WBATCH];
    int r_start[MAXR], r_prefix[MAXR + 1];
    int nranges, warp_cnt[8];
};

// shared by both kernels ------------------------------------------------------------------
struct TileGeom {
    int t0[3];    // tile origin (mesh index)
    int tv[3];    // valid width of the tile (16, or less at the upper mesh edge)
};

__device__ __forceinline__ int imod(int a, int n) { a %= n; return a < 0 ? a + n : a; }

// candidate ranges: the distinct bins {b-1, b, b+1} (periodic) in y and z, and in x the
// contiguous run b-1..b+1 split where it wraps
__device__ void tile_ranges(TileSmem& s, const int* __restrict__ cell_start, const int nb[3], int bx, int by, int bz)
{
    if (threadIdx.x == 0) {
        int n = 0, total = 0;
        int ys[3], zs[3], ny = 0, nz = 0;
        for (int o = -1; o <= 1; ++o) {
            int v = imod(by + o, nb[1]);
            bool dup = false;
            for (int k = 0; k < ny; ++k) dup |= (ys[k] == v);
            if (!dup) ys[ny++] = v;
            v = imod(bz + o, nb[2]);
            dup = false;
            for (int k = 0; k < nz; ++k) dup |= (zs[k] == v);
            if (!dup) zs[nz++] = v;
        }
        for (int iz = 0; iz < nz; ++iz)
            for (int iy = 0; iy < ny; ++iy) {
                const int row = (zs[iz] * nb[1] + ys[iy]) * nb[0];
                int lo[2], hi[2], np = 0;
                if (nb[0] <= 3) { lo[0] = 0; hi[0] = nb[0]; np = 1; }
                else if (bx == 0) { lo[0] = 0; hi[0] = 2; lo[1] = nb[0] - 1; hi[1] = nb[0]; np = 2; }
                else if (bx == nb[0] - 1) { lo[0] = bx - 1; hi[0] = nb[0]; lo[1] = 0; hi[1] = 1; np = 2; }
                else { lo[0] = bx - 1; hi[0] = bx + 2; np = 1; }
                for (int k = 0; k < np; ++k) {
                    const int a = cell_start[row + lo[k]], b = cell_start[row + hi[k]];
                    if (b > a) { s.r_start[n] = a; s.r_prefix[n] = total; total += b - a; ++n; }
                }
            }
        s.r_prefix[n] = total;
        s.nranges = n;
    }
    __syncthreads();
}

// phase A + B for one batch; returns the number of accepted particles (all threads)
template <bool SPREAD>
__device__ __forceinline__ int tile_batch(TileSmem& s, const WaveConst& wc, const TileGeom& tg, int base, int M,
                                          const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                                          const double* __restrict__ qs)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int P = wc.P;
    // ---- phase A
    bool ok = false;
    int pi = 0, dd[3] = {0, 0, 0};
    double uu[3] = {0, 0, 0}, qv = 0.0;
    const int c = base + tid;
    if (tid < WBATCH && c < M) {
        int r = 0;
        while (c >= s.r_prefix[r + 1]) ++r;
        pi = s.r_start[r] + (c - s.r_prefix[r]);
        const double pos[3] = {xs[pi], ys[pi], zs[pi]};
        ok = true;
        if (SPREAD) { qv = qs[pi]; ok = (qv != 0.0); }
#pragma unroll
        for (int dim = 0; dim < 3; ++dim) {
            const int ng = wc.Ng[dim];
            const double xd = pos[dim] * wc.inv_h[dim];
            const int i0 = min((int)xd, ng - 1);
            const int s0 = i0 - P / 2 + 1;  // first support index (reading A5, even P)
            const int dmod = imod(tg.t0[dim] - s0, ng);
            dd[dim] = dmod;
            uu[dim] = (double)s0 - xd;
            ok = ok && (dmod < P || dmod + tg.tv[dim] > ng);
        }
    }
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    if (lane == 0) s.warp_cnt[warp] = __popc(m);
    __syncthreads();
    int off = 0, nacc = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const int cw = s.warp_cnt[w];
        if (w < warp) off += cw;
        nacc += cw;
    }
    if (ok) {
        const int slot = off + __popc(m & ((1u << lane) - 1u));
        s.pidx[slot] = pi;
        s.q[slot] = qv;
#pragma unroll
        for (int dim = 0; dim < 3; ++dim) { s.d[slot][dim] = dd[dim]; s.ub[slot][dim] = uu[dim]; }
    }
    __syncthreads();
    // ---- phase B: weights of (slot, dim) into wt[slot][dim][0..16)
    for (int task = tid; task < nacc * 3; task += WTHREADS) {
        const int slot = task / 3, dim = task - slot * 3;
        const int ng = wc.Ng[dim], dsl = s.d[slot][dim], tv = tg.tv[dim];
        const double u0 = s.ub[slot][dim];
        double* w = s.wt[slot][dim];
#pragma unroll
        for (int j = 0; j < WT; ++j) w[j] = 0.0;
        double pw = exp(-wc.aw * u0 * u0);
        const double e1 = exp(-2.0 * wc.aw * u0);
        if (SPREAD && dim == 2) pw *= s.q[slot];
        for (int r = 0; r < P; ++r) {
            int j = r - dsl;
            if (j < 0) j += ng;
            if (j < tv) w[j] = pw * wc.G[r];
            pw *= e1;
        }
    }
    __syncthreads();
    return nacc;
}

// does the support of `slot` meet the brick starting at tile-local b0 of width bw (per dim)?
__device__ __forceinline__ bool brick_hit(const TileSmem& s, const WaveConst& wc, int slot, const int b0[3], const int bw[3])
{
    bool hit = true;
#pragma unroll
    for (int dim = 0; dim < 3; ++dim) {
        int db = s.d[slot][dim] + b0[dim];
        const int ng = wc.Ng[dim];
        if (db >= ng) db -= ng;
        hit = hit && (db < wc.P || db + bw[dim] > ng);
    }
    return hit;
}

__device__ __forceinline__ void tile_setup(const WaveConst& wc, const int nb[3], TileGeom& tg, int& bx, int& by, int& bz)
{
    int t = blockIdx.x;
    bx = t % nb[0]; t /= nb[0];
    by = t % nb[1]; bz = t / nb[1];
    tg.t0[0] = bx * WT; tg.t0[1] = by * WT; tg.t0[2] = bz * WT;
#pragma unroll
    for (int dim = 0; dim < 3; ++dim) tg.tv[dim] = min(WT, wc.Ng[dim] - tg.t0[dim]);
}

// ---------------------------------------------------------------- spread
__global__ void __launch_bounds__(WTHREADS, 2)
k_spread_tiles(WaveConst wc, int nbx, int nby, int nbz, const int* __restrict__ cell_start, const double* __restrict__ xs,
               const double* __restrict__ ys, const double* __restrict__ zs, const double* __restrict__ qs, double* __restrict__ grid)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& s = *reinterpret_cast<TileSmem*>(smem_raw);
    const int nb[3] = {nbx, nby, nbz};
    TileGeom tg;
    int bx, by, bz;
    tile_setup(wc, nb, tg, bx, by, bz);
    tile_ranges(s, cell_start, nb, bx, by, bz);
    const int M = s.r_prefix[s.nranges];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b0[3] = {(warp & 1) * 8, ((warp >> 1) & 1) * 8, (warp >> 2) * 8};
    const int bw[3] = {min(8, tg.tv[0] - b0[0]), min(8, tg.tv[1] - b0[1]), min(8, tg.tv[2] - b0[2])};
    const bool active = bw[0] > 0 && bw[1] > 0 && bw[2] > 0;
    const int px = b0[0] + (lane & 1) * 4, py = b0[1] + ((lane >> 1) & 1) * 4, pz = b0[2] + (lane >> 2);
    double acc[4][4];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[j][i] = 0.0;

    for (int base = 0; base < M; base += WBATCH) {
        const int nacc = tile_batch<true>(s, wc, tg, base, M, xs, ys, zs, qs);
        if (active) {
            for (int sb = 0; sb < nacc; sb += 32) {
                const int cand = sb + lane;
                unsigned mask = __ballot_sync(0xffffffffu, cand < nacc && brick_hit(s, wc, cand, b0, bw));
                while (mask) {
                    const int slot = sb + __ffs(mask) - 1;
                    mask &= mask - 1;
                    const double* wp = &s.wt[slot][0][0];
                    const double2 x01 = *reinterpret_cast<const double2*>(wp + px);
                    const double2 x23 = *reinterpret_cast<const double2*>(wp + px + 2);
                    const double2 y01 = *reinterpret_cast<const double2*>(wp + WT + py);
                    const double2 y23 = *reinterpret_cast<const double2*>(wp + WT + py + 2);
                    const double wzq = wp[2 * WT + pz];
                    const double cy[4] = {wzq * y01.x, wzq * y01.y, wzq * y23.x, wzq * y23.y};
                    const double wx[4] = {x01.x, x01.y, x23.x, x23.y};
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int i = 0; i < 4; ++i) acc[j][i] = fma(cy[j], wx[i], acc[j][i]);
                }
            }
        }
        __syncthreads();  // smem of this batch is recycled by the next
    }
    if (!active) return;
    const int gz = tg.t0[2] + pz;
    if (gz >= wc.Ng[2]) return;
    const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
    const int gx = tg.t0[0] + px;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int gy = tg.t0[1] + py + j;
        if (gy >= wc.Ng[1]) break;
        double* row = grid + ((size_t)gz * Ny + gy) * Nx + gx;
        if (gx + 3 < wc.Ng[0]) {
            *reinterpret_cast<double2*>(row) = make_double2(acc[j][0], acc[j][1]);
            *reinterpret_cast<double2*>(row + 2) = make_double2(acc[j][2], acc[j][3]);
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (gx + i < wc.Ng[0]) row[i] = acc[j][i];
        }
    }
}

// ---------------------------------------------------------------- gather
// reduce NV values per lane across the warp; afterwards lanes with (lane & (32/NV - 1)) == 0 hold the warp
// total of value number `id`
template <int NV>
__device__ __forceinline__ double transpose_reduce(double (&v)[NV], int lane, int& id)
{
    id = 0;
    int x = 16;
#pragma unroll
    for (int half = NV / 2; half >= 1; half >>= 1) {
        const bool up = (lane & x) != 0;
#pragma unroll
        for (int k = 0; k < half; ++k) {
            const double send = up ? v[k] : v[k + half];
            const double keep = up ? v[k + half] : v[k];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, send, x);
        }
        if (up) id += half;
        x >>= 1;
    }
    double r = v[0];
    for (; x >= 1; x >>= 1) r += __shfl_xor_sync(0xffffffffu, r, x);
    return r;
}

template <bool FIELD>
struct GatherCfg {
    static constexpr int NQ = FIELD ? 4 : 1;  // quantities per particle: psi (, Ex, Ey, Ez)
    static constexpr int G = FIELD ? 4 : 8;   // particles per butterfly
    static constexpr int NV = NQ * G;
};

template <bool FIELD>
__global__ void __launch_bounds__(WTHREADS, 2)
k_gather_tiles(WaveConst wc, int nbx, int nby, int nbz, const int* __restrict__ cell_start, const double* __restrict__ xs,
               const double* __restrict__ ys, const double* __restrict__ zs, const double* __restrict__ grid, double* __restrict__ psi,
               double* __restrict__ ex, double* __restrict__ ey, double* __restrict__ ez)
{
    using C = GatherCfg<FIELD>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& s = *reinterpret_cast<TileSmem*>(smem_raw);
    double* tot = reinterpret_cast<double*>(smem_raw + sizeof(TileSmem));  // [NQ][8][WBATCH]
    const int nb[3] = {nbx, nby, nbz};
    TileGeom tg;
    int bx, by, bz;
    tile_setup(wc, nb, tg, bx, by, bz);
    tile_ranges(s, cell_start, nb, bx, by, bz);
    const int M = s.r_prefix[s.nranges];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b0[3] = {(warp & 1) * 8, ((warp >> 1) & 1) * 8, (warp >> 2) * 8};
    const int bw[3] = {min(8, tg.tv[0] - b0[0]), min(8, tg.tv[1] - b0[1]), min(8, tg.tv[2] - b0[2])};
    const bool active = bw[0] > 0 && bw[1] > 0 && bw[2] > 0;
    const int px = b0[0] + (lane & 1) * 4, py = b0[1] + ((lane >> 1) & 1) * 4, pz = b0[2] + (lane >> 2);
    // the lane's 4x4 patch of H~ in registers (0 outside the mesh)
    double H[4][4];
    {
        const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
        const int gz = tg.t0[2] + pz, gx = tg.t0[0] + px;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int gy = tg.t0[1] + py + j;
            const bool rowok = M > 0 && gz < wc.Ng[2] && gy < wc.Ng[1];
            const double* row = grid + ((size_t)gz * Ny + gy) * Nx + gx;
            if (rowok && gx + 3 < wc.Ng[0]) {
                const double2 a = *reinterpret_cast<const double2*>(row), b = *reinterpret_cast<const double2*>(row + 2);
                H[j][0] = a.x; H[j][1] = a.y; H[j][2] = b.x; H[j][3] = b.y;
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) H[j][i] = (rowok && gx + i < wc.Ng[0]) ? row[i] : 0.0;
            }
        }
    }
    for (int base = 0; base < M; base += WBATCH) {
        const int nacc = tile_batch<false>(s, wc, tg, base, M, xs, ys, zs, nullptr);
        for (int k = tid; k < C::NQ * 8 * WBATCH; k += WTHREADS) tot[k] = 0.0;
        __syncthreads();
        if (active) {
            for (int sb = 0; sb < nacc; sb += 32) {
                const int cand = sb + lane;
                unsigned mask = __ballot_sync(0xffffffffu, cand < nacc && brick_hit(s, wc, cand, b0, bw));
                while (mask) {
                    double v[C::NV];
                    int slots[C::G];
#pragma unroll
                    for (int g = 0; g < C::G; ++g) {
                        if (mask) {
                            const int slot = sb + __ffs(mask) - 1;
                            mask &= mask - 1;
                            slots[g] = slot;
                            const double* wp = &s.wt[slot][0][0];
                            const double2 x01 = *reinterpret_cast<const double2*>(wp + px);
                            const double2 x23 = *reinterpret_cast<const double2*>(wp + px + 2);
                            const double2 y01 = *reinterpret_cast<const double2*>(wp + WT + py);
                            const double2 y23 = *reinterpret_cast<const double2*>(wp + WT + py + 2);
                            const double wz = wp[2 * WT + pz];
                            const double wx[4] = {x01.x, x01.y, x23.x, x23.y};
                            const double wy[4] = {y01.x, y01.y, y23.x, y23.y};
                            double t0[4];
#pragma unroll
                            for (int j = 0; j < 4; ++j)
                                t0[j] = fma(H[j][3], wx[3], fma(H[j][2], wx[2], fma(H[j][1], wx[1], H[j][0] * wx[0])));
                            const double s0 = fma(wy[3], t0[3], fma(wy[2], t0[2], fma(wy[1], t0[1], wy[0] * t0[0])));
                            if (!FIELD) {
                                v[g] = wz * s0;
                            } else {
                                // u = (mesh index - x/h) of the lane's points: ub + ((d + j) mod Ng)
                                double wxu[4], wyu[4];
#pragma unroll
                                for (int i = 0; i < 4; ++i) {
                                    int r = s.d[slot][0] + px + i;
                                    if (r >= wc.Ng[0]) r -= wc.Ng[0];
                                    wxu[i] = wx[i] * (s.ub[slot][0] + (double)r);
                                    r = s.d[slot][1] + py + i;
                                    if (r >= wc.Ng[1]) r -= wc.Ng[1];
                                    wyu[i] = wy[i] * (s.ub[slot][1] + (double)r);
                                }
                                int rz = s.d[slot][2] + pz;
                                if (rz >= wc.Ng[2]) rz -= wc.Ng[2];
                                const double uz = s.ub[slot][2] + (double)rz;
                                double t1[4];
#pragma unroll
                                for (int j = 0; j < 4; ++j)
                                    t1[j] = fma(H[j][3], wxu[3], fma(H[j][2], wxu[2], fma(H[j][1], wxu[1], H[j][0] * wxu[0])));
                                const double sx = fma(wy[3], t1[3], fma(wy[2], t1[2], fma(wy[1], t1[1], wy[0] * t1[0])));
                                const double sy = fma(wyu[3], t0[3], fma(wyu[2], t0[2], fma(wyu[1], t0[1], wyu[0] * t0[0])));
                                v[4 * g + 0] = wz * s0;
                                v[4 * g + 1] = wz * sx;
                                v[4 * g + 2] = wz * sy;
                                v[4 * g + 3] = wz * uz * s0;
                            }
                        } else {
                            slots[g] = -1;
#pragma unroll
                            for (int k = 0; k < C::NQ; ++k) v[C::NQ * g + k] = 0.0;
                        }
                    }
                    int id;
                    const double r = transpose_reduce<C::NV>(v, lane, id);
                    const int g = id / C::NQ, qn = id - g * C::NQ;
                    int slot = -1;
#pragma unroll
                    for (int k = 0; k < C::G; ++k)
                        if (k == g) slot = slots[k];
                    if ((lane & (32 / C::NV - 1)) == 0 && slot >= 0) tot[(qn * 8 + warp) * WBATCH + slot] = r;
                }
            }
        }
        __syncthreads();
        // sum the 8 bricks of the tile, one global atomic per particle and quantity
        for (int k = tid; k < C::NQ * nacc; k += WTHREADS) {
            const int qn = k / nacc, slot = k - qn * nacc;
            double sum = 0.0;
#pragma unroll
            for (int w = 0; w < 8; ++w) sum += tot[(qn * 8 + w) * WBATCH + slot];
            const int p = s.pidx[slot];
            if (qn == 0) atomicAdd(&psi[p], sum);
            else if (qn == 1) atomicAdd(&ex[p], -wc.grad_fac[0] * sum);  // E = -grad_alpha, dW/dx_alpha = +grad_fac u W
            else if (qn == 2) atomicAdd(&ey[p], -wc.grad_fac[1] * sum);
            else atomicAdd(&ez[p], -wc.grad_fac[2] * sum);
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- host
static size_t smem_spread() { return sizeof(TileSmem); }
template <bool FIELD> static size_t smem_gather() { return sizeof(TileSmem) + (size_t)GatherCfg<FIELD>::NQ * 8 * WBATCH * sizeof(double); }

int wave_tiles_init(pce_ctx* c)
{
    PCE_CUDA(c, cudaFuncSetAttribute(k_spread_tiles, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_spread()));
    PCE_CUDA(c, cudaFuncSetAttribute(k_gather_tiles<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_gather<false>()));
    PCE_CUDA(c, cudaFuncSetAttribute(k_gather_tiles<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_gather<true>()));
    return PCE_OK;
}

int wave_spread_tiles(pce_ctx* c, const Bins& b)
{
    PassTimer t(c, PASS_SPREAD);
    k_spread_tiles<<<b.ncell, WTHREADS, smem_spread(), c->st>>>(c->wk, b.nc[0], b.nc[1], b.nc[2], b.cell_start, b.xs, b.ys, b.zs, b.qs,
                                                                 c->grid);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

int wave_gather_tiles(pce_ctx* c, const Bins& b, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s)
{
    if (b.n == 0) return PCE_OK;
    PassTimer t(c, PASS_GATHER);
    PCE_CUDA(c, cudaMemsetAsync(psi_s, 0, (size_t)b.n * sizeof(double), c->st));
    if (field) {
        PCE_CUDA(c, cudaMemsetAsync(ex_s, 0, (size_t)b.n * sizeof(double), c->st));
        PCE_CUDA(c, cudaMemsetAsync(ey_s, 0, (size_t)b.n * sizeof(double), c->st));
        PCE_CUDA(c, cudaMemsetAsync(ez_s, 0, (size_t)b.n * sizeof(double), c->st));
        k_gather_tiles<true><<<b.ncell, WTHREADS, smem_gather<true>(), c->st>>>(c->wk, b.nc[0], b.nc[1], b.nc[2], b.cell_start, b.xs, b.ys,
                                                                                b.zs, c->grid, psi_s, ex_s, ey_s, ez_s);
    } else {
        k_gather_tiles<false><<<b.ncell, WTHREADS, smem_gather<false>(), c->st>>>(c->wk, b.nc[0], b.nc[1], b.nc[2], b.cell_start, b.xs,
                                                                                  b.ys, b.zs, c->grid, psi_s, nullptr, nullptr, nullptr);
    }
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
