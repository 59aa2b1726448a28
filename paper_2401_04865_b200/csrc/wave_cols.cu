// wave_cols.cu -- Gaussian spreading (eq. 25) and gather (eq. 27) on 8^3 bricks with
// CACHED hit lists, for meshes aligned with the brick lattice (N_g % 8 == 0, N_g - P >= 8; anything else: wave_bricks.cu).
//
// Positions are frozen for the ~30 operator applications of a Krylov solve, so everything that depends on
// positions only is built once per pce_set_positions:
//   * per particle a 64-byte hit record: first support index per dimension and the coefficients of the exp-free window
//     recurrence (see wave_bricks.cu), plus the particle's charge (rewritten per application);
//   * per brick COLUMN (bx, by) the list of particles whose (x, y) support meets the column, ordered by the first support
//     plane z_k (counting sort on the key (column, z_k), ties by particle slot: deterministic).  The hits of brick
//     (bx, by, bz) are the keys z_k in [8 bz - P + 1, 8 bz + 7] (cyclic): one or two contiguous runs of that list, found from
//     the key offsets alone -- no per-iteration candidate walk, ballot or queue.
// One warp owns a brick (persistent warps, bricks or chunks of crowded bricks handed out by a global counter).  Per batch of
// 32 hits: the records of the NEXT batch stream into shared memory with cp.async while the current batch runs; lane l turns
// record l into the 3 x 8 brick-local weights; the accumulation runs on the fp64 tensor path (mma.sync.m8n8k4.f64) exactly as
// in wave_bricks.cu.  Because the hits are ordered by z_k, the 4 (spread) or 8 (gather) hits of one mma group start at nearly
// the same plane: planes on which the whole group's window is zero are skipped (a per-hit live-plane mask, OR-ed per group),
// which removes most of the z part of the 27^3 brick envelope of a 20^3 support.
#include "pce_internal.h"

#include <cstdlib>

namespace {

constexpr int BR = 8;           // brick edge
constexpr int CW = 4;           // warps per CTA
constexpr int NTAB = 48 + 48;   // Gt[r + 8] = exp(-aw r^2), Ht[r + 8] = exp(-aw (2r + 1)), r = -8..39
constexpr int STRIDE_PSI = 26;  // doubles per hit in the weight table: 3 x 8 + 2 pad
constexpr int STRIDE_FLD = 50;  // with the field: 3 x (8 w + 8 w u) + 2 pad
constexpr int REC_BYTES = 64;

__device__ __forceinline__ int wrap_once(int d, int n) { if (d < 0) d += n; if (d >= n) d -= n; return d; }

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

struct ColGeom {
    int nbx, nby, nbz, Nz, P;
    int chunk;  // hits per work item (crowded bricks are split); 0: one item per brick
};

// ---------------------------------------------------------------- once per position update
// hit record of sorted particle i: window-recurrence coefficients (c_m, e1) per dimension, first support index per dimension,
// charge (filled per application), and u0 = s0 - x/h (field gather only) in a second array
__global__ void __launch_bounds__(256)
k_hit_records(int n, WaveConst wc, const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
              HitRec* __restrict__ rec, double4* __restrict__ u0o)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double pos[3] = {xs[i], ys[i], zs[i]};
    int sv[3];
    double uv[3];
    HitRec r;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double xd = pos[d] * wc.inv_h[d];
        const int i0 = min((int)xd, wc.Ng[d] - 1);
        const int s0 = i0 - wc.P / 2 + 1;  // first support index (reading A5, even P); may be negative
        const double u0 = (double)s0 - xd; // in (-P/2, -P/2 + 1]
        const int phi = (-s0) & (BR - 1);
        sv[d] = s0; uv[d] = u0;
        r.cf[d] = make_double2(exp(-wc.aw * u0 * (u0 + 2.0 * (phi - BR))), exp(-2.0 * wc.aw * u0));
    }
    r.s0[0] = (short)sv[0]; r.s0[1] = (short)sv[1]; r.s0[2] = (short)sv[2]; r.pad = 0;
    r.q = 0.0;
    rec[i] = r;
    u0o[i] = make_double4(uv[0], uv[1], uv[2], 0.0);
}

// keys (column, z_k): count, then (after the scan) fill; z_k = first support plane wrapped into [0, N_z)
template <bool FILL>
__global__ void __launch_bounds__(256)
k_col_keys(int n, ColGeom g, const HitRec* __restrict__ rec, int* __restrict__ cnt, const int* __restrict__ key_start, int* __restrict__ ent)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int4 s0 = make_int4(rec[i].s0[0], rec[i].s0[1], rec[i].s0[2], 0);
    const int fx = s0.x >> 3, lx = (s0.x + g.P - 1) >> 3, fy = s0.y >> 3, ly = (s0.y + g.P - 1) >> 3;  // >> 3: floor for negatives too
    const int zk = s0.z < 0 ? s0.z + g.Nz : s0.z;
    for (int iy = fy; iy <= ly; ++iy) {
        const int by = wrap_once(iy, g.nby);
        for (int ix = fx; ix <= lx; ++ix) {
            const int bx = wrap_once(ix, g.nbx);
            const int key = (by * g.nbx + bx) * g.Nz + zk;
            const int slot = atomicAdd(&cnt[key], 1);
            if (FILL) ent[key_start[key] + slot] = i;
        }
    }
}

// order the entries of every key by particle slot (the atomic fill order is arbitrary): small keys one thread each
// (insertion sort), larger keys one warp each (rank by counting through shared memory, or in place for huge keys)
__global__ void __launch_bounds__(256)
k_col_sort_small(int nkeys, const int* __restrict__ key_start, int* __restrict__ ent, int* __restrict__ big_list)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nkeys) return;
    const int b = key_start[k], n = key_start[k + 1] - b;
    if (n < 2) return;
    if (n > 8) { big_list[atomicAdd(&big_list[nkeys], 1)] = k; return; }  // left to k_col_sort_big (list order is irrelevant)
    int v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = (i < n) ? ent[b + i] : 0x7fffffff;
#pragma unroll
    for (int i = 1; i < 8; ++i) {
#pragma unroll
        for (int j = i; j > 0; --j) {
            const int lo = min(v[j - 1], v[j]), hi = max(v[j - 1], v[j]);
            v[j - 1] = lo; v[j] = hi;
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i)
        if (i < n) ent[b + i] = v[i];
}

constexpr int SORT_CAP = 1024;  // entries of one key sorted through shared memory by one warp
__global__ void __launch_bounds__(128)
k_col_sort_big(int nkeys, const int* __restrict__ key_start, int* __restrict__ ent, const int* __restrict__ big_list)
{
    __shared__ int buf[4][SORT_CAP];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nbig = big_list[nkeys];
    for (int e = blockIdx.x * 4 + warp; e < nbig; e += gridDim.x * 4) {
        const int k = big_list[e];
        const int b = key_start[k], n = key_start[k + 1] - b;
        if (n <= SORT_CAP) {
            int* s = buf[warp];
            for (int i = lane; i < n; i += 32) s[i] = ent[b + i];
            __syncwarp();
            for (int i = lane; i < n; i += 32) {
                const int mine = s[i];
                int rank = 0;
                for (int j = 0; j < n; ++j) rank += (s[j] < mine);  // entries of a key are distinct particles
                ent[b + rank] = mine;
            }
            __syncwarp();
        } else {  // odd-even transposition in place (pathological crowding only)
            for (int phase = 0; phase < n; ++phase) {
                for (int i = (phase & 1) + 2 * lane; i + 1 < n; i += 64) {
                    const int x = ent[b + i], y = ent[b + i + 1];
                    if (x > y) { ent[b + i] = y; ent[b + i + 1] = x; }
                }
                __syncwarp();
            }
        }
    }
}

// work items: brick b has max(1, ceil(hits / chunk)) items (empty bricks still write their zeros in the spread)
__device__ __forceinline__ void brick_runs(const ColGeom& g, const int* __restrict__ key_start, int brick, int& a0, int& n0, int& a1, int& n1)
{
    const int ncol = g.nbx * g.nby;
    const int col = brick % ncol, bz = brick / ncol;
    const int base = col * g.Nz;
    const int lo = BR * bz - g.P + 1, hi = BR * bz + BR - 1;  // z_k range (hi < N_z always)
    if (lo >= 0) {
        a0 = key_start[base + lo]; n0 = key_start[base + hi + 1] - a0; a1 = 0; n1 = 0;
    } else {  // wrapped part first: those supports start "before" the brick
        a0 = key_start[base + lo + g.Nz]; n0 = key_start[base + g.Nz] - a0;
        a1 = key_start[base]; n1 = key_start[base + hi + 1] - a1;
    }
}

__global__ void __launch_bounds__(256)
k_item_count(int nbrick, ColGeom g, const int* __restrict__ key_start, int* __restrict__ item_start)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > nbrick) return;
    int v = 0;
    if (b < nbrick) {
        int a0, n0, a1, n1;
        brick_runs(g, key_start, b, a0, n0, a1, n1);
        const int nh = n0 + n1;
        v = (g.chunk > 0 && nh > g.chunk) ? (nh + g.chunk - 1) / g.chunk : 1;
    }
    item_start[b] = v;
}

__global__ void __launch_bounds__(256)
k_item_fill(int nbrick, const int* __restrict__ item_start, int2* __restrict__ items)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbrick) return;
    const int s = item_start[b], e = item_start[b + 1];
    for (int i = s; i < e; ++i) items[i] = make_int2(b, i - s);
}

// ---------------------------------------------------------------- shared pieces of the two kernels
template <int STRIDE>
struct alignas(16) WarpSmem {
    double wt[32 * STRIDE];                 // brick-local weights of the current batch
    unsigned char rec[32 * REC_BYTES];      // hit records of the batch being loaded (16-byte chunks XOR-swizzled by hit index)
    unsigned char mask[16];                 // live planes of each mma group of the current batch
};

struct Item {
    int brick, b0[3];
    int a0, n0, a1;   // runs of the column list
    int h0, h1;       // hits [h0, h1) of the brick handled by this item
    int nh_brick, nitems, chunk_id;
};

__device__ __forceinline__ bool next_item(const ColGeom& g, const int* __restrict__ key_start, const int2* __restrict__ items, int n_items,
                                          int* __restrict__ work_ctr, int lane, Item& it)
{
    int id = 0;
    if (lane == 0) id = atomicAdd(work_ctr, 1);
    id = __shfl_sync(0xffffffffu, id, 0);
    if (id >= n_items) return false;
    int brick = id, chunk_id = 0;
    if (items) { const int2 v = items[id]; brick = v.x; chunk_id = v.y; }
    int a0, n0, a1, n1;
    brick_runs(g, key_start, brick, a0, n0, a1, n1);
    it.brick = brick; it.chunk_id = chunk_id;
    int t = brick;
    it.b0[0] = (t % g.nbx) * BR; t /= g.nbx;
    it.b0[1] = (t % g.nby) * BR; it.b0[2] = (t / g.nby) * BR;
    it.a0 = a0; it.n0 = n0; it.a1 = a1;
    it.nh_brick = n0 + n1;
    if (g.chunk > 0 && it.nh_brick > g.chunk) {
        it.nitems = (it.nh_brick + g.chunk - 1) / g.chunk;
        it.h0 = chunk_id * g.chunk;
        it.h1 = min(it.nh_brick, it.h0 + g.chunk);
    } else {
        it.nitems = 1; it.h0 = 0; it.h1 = it.nh_brick;
    }
    return true;
}

// particle slot of hit h of the brick (h < nh_brick), or -1
__device__ __forceinline__ int hit_slot(const Item& it, const int* __restrict__ ent, int h)
{
    if (h >= it.h1) return -1;
    return ent[h < it.n0 ? it.a0 + h : it.a1 + (h - it.n0)];
}

// stream the records of 32 hits (slot p per lane, -1: none) into the warp's buffer: instruction k moves records 8k..8k+7 whole
// (4 lanes x 16 bytes each), chunk c of record r lands at r*64 + ((c ^ ((r >> 1) & 3)) * 16): conflict-free 16-byte reads per lane later
__device__ __forceinline__ void prefetch_records(unsigned char* __restrict__ rbuf, const HitRec* __restrict__ rec, int p, int lane)
{
    const int c = lane & 3;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int r = 8 * k + (lane >> 2);
        const int pr = __shfl_sync(0xffffffffu, p, r);
        if (pr >= 0) cp_async16(rbuf + r * REC_BYTES + ((c ^ ((r >> 1) & 3)) << 4), reinterpret_cast<const unsigned char*>(rec + pr) + (c << 4));
    }
    cp_async_commit();
}

__device__ __forceinline__ double4 ld_u0(const double4* __restrict__ u0g, int p)
{
    const double2 a = __ldg(reinterpret_cast<const double2*>(u0g + p)), b = __ldg(reinterpret_cast<const double2*>(u0g + p) + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

template <class T>
__device__ __forceinline__ T rec_chunk(const unsigned char* rbuf, int r, int c)
{
    return *reinterpret_cast<const T*>(rbuf + r * REC_BYTES + ((c ^ ((r >> 1) & 3)) << 4));
}

// the 8 brick-local window weights of one hit in one dimension (0 outside the support) and, with FIELD, the weights times
// u = (mesh index - x/h); returns the mask of live brick-local points.  cf = (c_m, e1): weight factor at support index phi - 8
// and exp(-2 aw u0); tab = [Gt | Ht].
template <bool FIELD>
__device__ __forceinline__ unsigned brick_weights(int P, const double* __restrict__ tab, int b0, int ng, int s0, const double2 cf, double u0,
                                                  double scale, double* __restrict__ w)
{
    int r0 = b0 - s0;                   // support index of brick-local point 0, brought into -7 .. P-1
    if (r0 >= P) r0 -= ng;
    if (r0 < -7) r0 += ng;
    const int phi = (-s0) & (BR - 1);
    const int m1 = ((r0 - phi) >> 3) + 1;  // 0 .. 4: r0 = phi - 8 + 8 m1
    const double e2 = cf.y * cf.y, e4 = e2 * e2, e8 = e4 * e4, e16 = e8 * e8;
    double pm = (m1 & 1) ? e8 : 1.0;       // e8^m1
    if (m1 & 2) pm *= e16;
    if (m1 & 4) pm = e16 * e16;
    double pw = cf.x * pm * tab[r0 + 8] * scale;
    double t = cf.y * tab[48 + r0 + 8];
    const double g2 = tab[9] * tab[9];  // exp(-2 aw)
    // live points j: 0 <= r0 + j < P
    const int lo = max(0, -r0), hi = min(BR, P - r0);
    const unsigned live = ((1u << hi) - 1u) & ~((1u << lo) - 1u);
    double v[BR], vu[BR];
#pragma unroll
    for (int j = 0; j < BR; ++j) {
        v[j] = (live & (1u << j)) ? pw : 0.0;
        if (FIELD) vu[j] = v[j] * (u0 + (double)(r0 + j));
        pw *= t;
        t *= g2;
    }
#pragma unroll
    for (int j = 0; j < BR; j += 2) *reinterpret_cast<double2*>(w + j) = make_double2(v[j], v[j + 1]);
    if (FIELD) {
#pragma unroll
        for (int j = 0; j < BR; j += 2) *reinterpret_cast<double2*>(w + BR + j) = make_double2(vu[j], vu[j + 1]);
    }
    return live;
}

__device__ __forceinline__ void load_tables(const WaveConst& wc, double* tab)
{
    for (int k = threadIdx.x; k < NTAB; k += blockDim.x) {
        const int r = (k < 48 ? k : k - 48) - 8;
        tab[k] = (k < 48) ? exp(-wc.aw * (double)(r * r)) : exp(-wc.aw * (double)(2 * r + 1));
    }
    __syncthreads();
}

// weights of the nh hits whose records sit in the warp's buffer (one hit per lane): table rows + live-plane masks
template <bool FIELD, int STRIDE, int DW, int GROUP>
__device__ __forceinline__ void batch_weights(const WaveConst& wc, const double* __restrict__ tab, const Item& it, WarpSmem<STRIDE>& s, int nh,
                                              int lane, bool use_q, double4 u0v)
{
    unsigned zmask = 0;
    if (lane < nh) {
        const double2 sq = rec_chunk<double2>(s.rec, lane, 3);   // (s0 as 3 x int16, charge)
        const int shi = __double2hiint(sq.x), slo = __double2loint(sq.x);
        const int4 s0 = make_int4((int)(short)(slo & 0xffff), slo >> 16, (int)(short)(shi & 0xffff), 0);
        const double q = use_q ? sq.y : 1.0;
        double* w = s.wt + lane * STRIDE;
        const int sv[3] = {s0.x, s0.y, s0.z};
        const double uv[3] = {u0v.x, u0v.y, u0v.z};
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const unsigned lv = brick_weights<FIELD>(wc.P, tab, it.b0[d], wc.Ng[d], sv[d], rec_chunk<double2>(s.rec, lane, d), uv[d],
                                                     d == 2 ? q : 1.0, w + DW * d);
            if (d == 2) zmask = lv;
        }
    }
    // planes live for any hit of an mma group (GROUP = 4 hits in the spread, 8 in the gather): one byte per group
    zmask |= __shfl_xor_sync(0xffffffffu, zmask, 1);
    zmask |= __shfl_xor_sync(0xffffffffu, zmask, 2);
    if (GROUP == 8) zmask |= __shfl_xor_sync(0xffffffffu, zmask, 4);
    // stored per PAIR of planes (bit k: plane 2k or 2k + 1 live): the kernels skip dead pairs by a jump table, because a
    // predicated-off DMMA occupies the fp64 datapath exactly like a live one (measured) and short branches are if-converted
    const unsigned pm = (zmask | (zmask >> 1)) & 0x55u;
    if ((lane & (GROUP - 1)) == 0) s.mask[lane / GROUP] = (unsigned char)((pm & 1u) | ((pm >> 1) & 2u) | ((pm >> 2) & 4u) | ((pm >> 3) & 8u));
    __syncwarp();
}

// ---------------------------------------------------------------- spread
// H_z[y][x] = sum_h (wy_h[y] q_h wz_h[z]) wx_h[x] per plane z of the brick, four hits per fp64 mma, planes dead for the whole
// group skipped.  A brick split into several items (crowded bricks on small meshes) is combined deterministically: every item
// stores its partial brick in scratch, the item that arrives last adds them in item order and writes the mesh.
__global__ void __launch_bounds__(CW * 32, 6)
k_spread_cols(WaveConst wc, ColGeom g, const int* __restrict__ key_start, const int* __restrict__ ent, const int2* __restrict__ items,
              int n_items, const int* __restrict__ item_start, const HitRec* __restrict__ rec, double* __restrict__ grid,
              double* __restrict__ scratch, int* __restrict__ arrive, int* __restrict__ work_ctr, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    if (items) n_items = item_start[g.nbx * g.nby * g.nbz];  // chunked binnings: the item count lives on the device
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* tab = reinterpret_cast<double*>(smem_raw);
    WarpSmem<STRIDE_PSI>* sm = reinterpret_cast<WarpSmem<STRIDE_PSI>*>(smem_raw + NTAB * sizeof(double));
    load_tables(wc, tab);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem<STRIDE_PSI>& s = sm[warp];
    const int gq = lane >> 2, t = lane & 3;  // mma fragment coordinates
    const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
    Item it;
    while (next_item(g, key_start, items, n_items, work_ctr, lane, it)) {
        double acc[BR][2];  // plane z: H[z][y = gq][x = 2t, 2t + 1]
#pragma unroll
        for (int z = 0; z < BR; ++z) { acc[z][0] = 0.0; acc[z][1] = 0.0; }
        // software pipeline: slot indices two batches ahead, records one batch ahead
        int p_cur = hit_slot(it, ent, it.h0 + lane);
        prefetch_records(s.rec, rec, p_cur, lane);
        int p_next = hit_slot(it, ent, it.h0 + 32 + lane);
        for (int hb = it.h0; hb < it.h1; hb += 32) {
            const int nh = min(32, it.h1 - hb);
            cp_async_wait_all();
            __syncwarp();
            batch_weights<false, STRIDE_PSI, BR, 4>(wc, tab, it, s, nh, lane, true, make_double4(0, 0, 0, 0));
            if (hb + 32 < it.h1) {  // the records are consumed: start the next batch's
                prefetch_records(s.rec, rec, p_next, lane);
                p_next = hit_slot(it, ent, hb + 64 + lane);
            }
            for (int sb = 0; sb < nh; sb += 4) {
                const bool live = sb + t < nh;
                const double* w = s.wt + (live ? sb + t : 0) * STRIDE_PSI;
                const double bx = live ? w[gq] : 0.0;        // B[t][gq] = wx_h[x = gq]
                const double ay = live ? w[BR + gq] : 0.0;   // wy_h[y = gq]
                const unsigned m = s.mask[sb >> 2];          // plane pairs live for any hit of the group
#define SPREAD_PAIR(z)                                                                                   \
    {                                                                                                    \
        const double2 wz = *reinterpret_cast<const double2*>(w + 2 * BR + (z)); /* q_h wz_h[z], [z + 1] */ \
        dmma884(acc[z][0], acc[z][1], ay * wz.x, bx);                                                    \
        dmma884(acc[(z) + 1][0], acc[(z) + 1][1], ay * wz.y, bx);                                        \
    }
                switch (m) {  // the live pairs of a group are contiguous (supports are); anything else: all pairs (dead weights are 0)
                    case 0x1: SPREAD_PAIR(0) break;
                    case 0x3: SPREAD_PAIR(0) SPREAD_PAIR(2) break;
                    case 0x7: SPREAD_PAIR(0) SPREAD_PAIR(2) SPREAD_PAIR(4) break;
                    case 0x8: SPREAD_PAIR(6) break;
                    case 0xc: SPREAD_PAIR(4) SPREAD_PAIR(6) break;
                    case 0xe: SPREAD_PAIR(2) SPREAD_PAIR(4) SPREAD_PAIR(6) break;
                    case 0x2: SPREAD_PAIR(2) break;
                    case 0x4: SPREAD_PAIR(4) break;
                    case 0x6: SPREAD_PAIR(2) SPREAD_PAIR(4) break;
                    case 0x0: break;
                    default: SPREAD_PAIR(0) SPREAD_PAIR(2) SPREAD_PAIR(4) SPREAD_PAIR(6) break;
                }
#undef SPREAD_PAIR
            }
            __syncwarp();
        }
        const int gx = it.b0[0] + 2 * t, gy = it.b0[1] + gq;
        if (it.nitems > 1) {
            // partial brick -> scratch; the last of the brick's items to arrive sums them in item order
            const int first = item_start[it.brick];
            double* mine = scratch + (size_t)(first + it.chunk_id) * 512;
#pragma unroll
            for (int z = 0; z < BR; ++z) *reinterpret_cast<double2*>(mine + z * 64 + gq * 8 + 2 * t) = make_double2(acc[z][0], acc[z][1]);
            __threadfence();
            __syncwarp();
            int prev = 0;
            if (lane == 0) prev = atomicAdd(&arrive[it.brick], 1);
            prev = __shfl_sync(0xffffffffu, prev, 0);
            if (prev != it.nitems - 1) continue;
            if (lane == 0) arrive[it.brick] = 0;
            __threadfence();
#pragma unroll
            for (int z = 0; z < BR; ++z) { acc[z][0] = 0.0; acc[z][1] = 0.0; }
            for (int k = 0; k < it.nitems; ++k) {
                const double* part = scratch + (size_t)(first + k) * 512;
#pragma unroll
                for (int z = 0; z < BR; ++z) {
                    const double2 v = __ldcg(reinterpret_cast<const double2*>(part + z * 64 + gq * 8 + 2 * t));
                    acc[z][0] += v.x; acc[z][1] += v.y;
                }
            }
        }
#pragma unroll
        for (int z = 0; z < BR; ++z) {
            double* row = grid + ((size_t)(it.b0[2] + z) * Ny + gy) * Nx + gx;
            *reinterpret_cast<double2*>(row) = make_double2(acc[z][0], acc[z][1]);
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------- gather
// T_z[h][x] = sum_y wy_h[y] H~_z[y][x] (two fp64 mma k-steps per plane and 8 hits, the brick of H~ held in registers as the B
// operand), U[h][x] += wz_h[z] T_z[h][x], psi_h += sum_x wx_h[x] U[h][x]; one atomicAdd per hit, item and quantity.  With the
// field the window-gradient sums (reading A3) reuse T_z with wz u_z and wx u_x and need a second contraction with wy u_y.
template <bool FIELD>
__global__ void __launch_bounds__(CW * 32, FIELD ? 3 : 6)
k_gather_cols(WaveConst wc, ColGeom g, const int* __restrict__ key_start, const int* __restrict__ ent, const int2* __restrict__ items,
              int n_items, const int* __restrict__ item_start, const HitRec* __restrict__ rec, const double4* __restrict__ u0g,
              const double* __restrict__ grid,
              double* __restrict__ psi, double* __restrict__ ex, double* __restrict__ ey, double* __restrict__ ez,
              int* __restrict__ work_ctr, const int* __restrict__ skip, const int* __restrict__ pair_start, double* __restrict__ part,
              long long part_stride)
{
    // pair_start != nullptr (PCE_FLAG_DETERMINISTIC): the contribution of hit h of brick b goes to part[pair_start[b] + h] (one
    // plain store per pair and quantity) and k_gather_finish adds each particle's pairs in a fixed order; else one atomicAdd
    if (skip && *skip) return;
    if (items) n_items = item_start[g.nbx * g.nby * g.nbz];
    constexpr int STRIDE = FIELD ? STRIDE_FLD : STRIDE_PSI;
    constexpr int DW = FIELD ? 2 * BR : BR;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* tab = reinterpret_cast<double*>(smem_raw);
    WarpSmem<STRIDE>* sm = reinterpret_cast<WarpSmem<STRIDE>*>(smem_raw + NTAB * sizeof(double));
    load_tables(wc, tab);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem<STRIDE>& s = sm[warp];
    const int gq = lane >> 2, t = lane & 3;
    const size_t Nx = wc.Ng[0], Ny = wc.Ng[1];
    Item it;
    while (next_item(g, key_start, items, n_items, work_ctr, lane, it)) {
        if (it.h1 <= it.h0) continue;
        int p_cur = hit_slot(it, ent, it.h0 + lane);
        prefetch_records(s.rec, rec, p_cur, lane);
        int p_next = hit_slot(it, ent, it.h0 + 32 + lane);
        double4 u_cur = make_double4(0, 0, 0, 0), u_next = u_cur;
        if (FIELD) {
            if (p_cur >= 0) u_cur = ld_u0(u0g, p_cur);
            if (p_next >= 0) u_next = ld_u0(u0g, p_next);
        }
        // B operands: H[z][0] = H~[z][y = t][x = gq], H[z][1] = H~[z][y = t + 4][x = gq]
        double H[BR][2];
#pragma unroll
        for (int z = 0; z < BR; ++z) {
            const double* pl = grid + ((size_t)(it.b0[2] + z) * Ny + it.b0[1]) * Nx + it.b0[0] + gq;
            H[z][0] = pl[(size_t)t * Nx];
            H[z][1] = pl[(size_t)(t + 4) * Nx];
        }
        for (int hb = it.h0; hb < it.h1; hb += 32) {
            const int nh = min(32, it.h1 - hb);
            cp_async_wait_all();
            __syncwarp();
            batch_weights<FIELD, STRIDE, DW, 8>(wc, tab, it, s, nh, lane, false, u_cur);
            const int p_mine = p_cur;  // slot of hit hb + lane (output index)
            const long long pair0 = pair_start ? (long long)pair_start[it.brick] + hb : 0;
            p_cur = p_next; u_cur = u_next;
            if (hb + 32 < it.h1) {
                prefetch_records(s.rec, rec, p_next, lane);
                p_next = hit_slot(it, ent, hb + 64 + lane);
                if (FIELD) u_next = (p_next >= 0) ? ld_u0(u0g, p_next) : make_double4(0, 0, 0, 0);
            }
            for (int sb = 0; sb < nh; sb += 8) {
                const int hr = sb + gq;
                const bool live = hr < nh;
                const double* w = s.wt + (live ? hr : 0) * STRIDE;
                const double a0 = live ? w[DW + t] : 0.0, a1 = live ? w[DW + t + 4] : 0.0;  // wy_h[y]
                const double2 wx2 = *reinterpret_cast<const double2*>(w + 2 * t);           // wx_h[2t], [2t + 1]
                const unsigned m = s.mask[sb >> 3];  // plane pairs live for any hit of the group
                const int po = __shfl_sync(0xffffffffu, p_mine, hr & 31);
                if (!FIELD) {
                    double u0 = 0.0, u1 = 0.0;
#define GATHER_PAIR(z)                                                                       \
    {                                                                                        \
        const double2 wz = *reinterpret_cast<const double2*>(w + 2 * DW + (z));              \
        double t0 = 0.0, t1 = 0.0, s0 = 0.0, s1 = 0.0;                                       \
        dmma884(t0, t1, a0, H[z][0]);                                                        \
        dmma884(t0, t1, a1, H[z][1]);                                                        \
        dmma884(s0, s1, a0, H[(z) + 1][0]);                                                  \
        dmma884(s0, s1, a1, H[(z) + 1][1]);                                                  \
        u0 = fma(wz.x, t0, u0); u1 = fma(wz.x, t1, u1);                                      \
        u0 = fma(wz.y, s0, u0); u1 = fma(wz.y, s1, u1);                                      \
    }
                    switch (m) {  // live plane pairs of the group (contiguous); anything else: all pairs (dead weights are 0)
                        case 0x1: GATHER_PAIR(0) break;
                        case 0x3: GATHER_PAIR(0) GATHER_PAIR(2) break;
                        case 0x7: GATHER_PAIR(0) GATHER_PAIR(2) GATHER_PAIR(4) break;
                        case 0x8: GATHER_PAIR(6) break;
                        case 0xc: GATHER_PAIR(4) GATHER_PAIR(6) break;
                        case 0xe: GATHER_PAIR(2) GATHER_PAIR(4) GATHER_PAIR(6) break;
                        case 0x2: GATHER_PAIR(2) break;
                        case 0x4: GATHER_PAIR(4) break;
                        case 0x6: GATHER_PAIR(2) GATHER_PAIR(4) break;
                        case 0x0: break;
                        default: GATHER_PAIR(0) GATHER_PAIR(2) GATHER_PAIR(4) GATHER_PAIR(6) break;
                    }
#undef GATHER_PAIR
                    double r = fma(wx2.y, u1, wx2.x * u0);
                    r += __shfl_xor_sync(0xffffffffu, r, 1);
                    r += __shfl_xor_sync(0xffffffffu, r, 2);
                    if (live && t == 0) {
                        if (pair_start) part[pair0 + hr] = r;
                        else atomicAdd(&psi[po], r);
                    }
                } else {
                    const double b0 = live ? w[DW + BR + t] : 0.0, b1 = live ? w[DW + BR + t + 4] : 0.0;  // wy u_y
                    const double2 wxu2 = *reinterpret_cast<const double2*>(w + BR + 2 * t);               // wx u_x
                    double u0 = 0.0, u1 = 0.0, uz0 = 0.0, uz1 = 0.0, uy0 = 0.0, uy1 = 0.0;
#define GATHER_PLANE_F(z)                                                                    \
    {                                                                                        \
        const double wz = w[2 * DW + (z)], wzu = w[2 * DW + BR + (z)];                       \
        double t0 = 0.0, t1 = 0.0, v0 = 0.0, v1 = 0.0;                                       \
        dmma884(t0, t1, a0, H[z][0]);                                                        \
        dmma884(t0, t1, a1, H[z][1]);                                                        \
        dmma884(v0, v1, b0, H[z][0]);                                                        \
        dmma884(v0, v1, b1, H[z][1]);                                                        \
        u0 = fma(wz, t0, u0); u1 = fma(wz, t1, u1);                                          \
        uz0 = fma(wzu, t0, uz0); uz1 = fma(wzu, t1, uz1);                                    \
        uy0 = fma(wz, v0, uy0); uy1 = fma(wz, v1, uy1);                                      \
    }
#define GATHER_PAIR_F(z) GATHER_PLANE_F(z) GATHER_PLANE_F((z) + 1)
                    switch (m) {
                        case 0x1: GATHER_PAIR_F(0) break;
                        case 0x3: GATHER_PAIR_F(0) GATHER_PAIR_F(2) break;
                        case 0x7: GATHER_PAIR_F(0) GATHER_PAIR_F(2) GATHER_PAIR_F(4) break;
                        case 0x8: GATHER_PAIR_F(6) break;
                        case 0xc: GATHER_PAIR_F(4) GATHER_PAIR_F(6) break;
                        case 0xe: GATHER_PAIR_F(2) GATHER_PAIR_F(4) GATHER_PAIR_F(6) break;
                        case 0x2: GATHER_PAIR_F(2) break;
                        case 0x4: GATHER_PAIR_F(4) break;
                        case 0x6: GATHER_PAIR_F(2) GATHER_PAIR_F(4) break;
                        case 0x0: break;
                        default: GATHER_PAIR_F(0) GATHER_PAIR_F(2) GATHER_PAIR_F(4) GATHER_PAIR_F(6) break;
                    }
#undef GATHER_PAIR_F
#undef GATHER_PLANE_F
                    double r0 = fma(wx2.y, u1, wx2.x * u0);      // psi
                    double r1 = fma(wxu2.y, u1, wxu2.x * u0);    // sum W u_x H
                    double r2 = fma(wx2.y, uy1, wx2.x * uy0);    // sum W u_y H
                    double r3 = fma(wx2.y, uz1, wx2.x * uz0);    // sum W u_z H
                    r0 += __shfl_xor_sync(0xffffffffu, r0, 1); r1 += __shfl_xor_sync(0xffffffffu, r1, 1);
                    r2 += __shfl_xor_sync(0xffffffffu, r2, 1); r3 += __shfl_xor_sync(0xffffffffu, r3, 1);
                    r0 += __shfl_xor_sync(0xffffffffu, r0, 2); r1 += __shfl_xor_sync(0xffffffffu, r1, 2);
                    r2 += __shfl_xor_sync(0xffffffffu, r2, 2); r3 += __shfl_xor_sync(0xffffffffu, r3, 2);
                    if (live) {  // E = -grad_a, dW/dx_a = +grad_fac u W; lane t issues quantity t
                        const double val = (t == 0) ? r0 : (t == 1) ? -wc.grad_fac[0] * r1 : (t == 2) ? -wc.grad_fac[1] * r2 : -wc.grad_fac[2] * r3;
                        if (pair_start) part[(long long)t * part_stride + pair0 + hr] = val;
                        else atomicAdd((t == 0) ? &psi[po] : (t == 1) ? &ex[po] : (t == 2) ? &ey[po] : &ez[po], val);
                    }
                }
            }
            __syncwarp();
        }
    }
}

// ---------------------------------------------------------------- deterministic gather (PCE_FLAG_DETERMINISTIC)
// pairs (brick, hit) are numbered pair_start[brick] + h; particle p meets the bricks (fx + i, fy + j, fz + k) of its support in a
// fixed enumeration, so the slot of a pair in the particle's list follows from the brick coordinates alone: no atomics, no sort
__global__ void __launch_bounds__(256)
k_pair_count(int nbrick, ColGeom g, const int* __restrict__ key_start, int* __restrict__ pair_start)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > nbrick) return;
    int v = 0;
    if (b < nbrick) {
        int a0, n0, a1, n1;
        brick_runs(g, key_start, b, a0, n0, a1, n1);
        v = n0 + n1;
    }
    pair_start[b] = v;
}

__device__ __forceinline__ void brick_span(int s0, int P, int& f, int& cnt)
{
    f = s0 >> 3;  // floor for negatives too
    cnt = ((s0 + P - 1) >> 3) - f + 1;
}

__global__ void __launch_bounds__(256)
k_inv_count(int n, int P, const HitRec* __restrict__ rec, int* __restrict__ inv_ptr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    int v = 0;
    if (i < n) {
        const int4 s0 = make_int4(rec[i].s0[0], rec[i].s0[1], rec[i].s0[2], 0);
        int f, cx, cy, cz;
        brick_span(s0.x, P, f, cx); brick_span(s0.y, P, f, cy); brick_span(s0.z, P, f, cz);
        v = cx * cy * cz;
    }
    inv_ptr[i] = v;
}

// one warp per brick: pair (brick, h) -> slot in the list of its particle
__global__ void __launch_bounds__(256)
k_inv_fill(int nbrick, ColGeom g, const int* __restrict__ key_start, const int* __restrict__ ent, const HitRec* __restrict__ rec,
           const int* __restrict__ pair_start, const int* __restrict__ inv_ptr, int* __restrict__ inv_list)
{
    const int b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (b >= nbrick) return;
    int a0, n0, a1, n1;
    brick_runs(g, key_start, b, a0, n0, a1, n1);
    int t = b;
    const int bx = t % g.nbx; t /= g.nbx;
    const int by = t % g.nby, bz = t / g.nby;
    const int base = pair_start[b];
    for (int h = lane; h < n0 + n1; h += 32) {
        const int p = ent[h < n0 ? a0 + h : a1 + (h - n0)];
        const int4 s0 = make_int4(rec[p].s0[0], rec[p].s0[1], rec[p].s0[2], 0);
        int fx, fy, fz, cx, cy, cz;
        brick_span(s0.x, g.P, fx, cx); brick_span(s0.y, g.P, fy, cy); brick_span(s0.z, g.P, fz, cz);
        int dx = (bx - fx) % g.nbx, dy = (by - fy) % g.nby, dz = (bz - fz) % g.nbz;
        if (dx < 0) dx += g.nbx;
        if (dy < 0) dy += g.nby;
        if (dz < 0) dz += g.nbz;
        inv_list[inv_ptr[p] + (dz * cy + dy) * cx + dx] = base + h;
    }
}

// psi[p] = sum of the particle's pair contributions, in list order (fixed: bit-reproducible)
__global__ void __launch_bounds__(256)
k_gather_finish(int n, int nq, const int* __restrict__ inv_ptr, const int* __restrict__ inv_list, const double* __restrict__ part,
                long long part_stride, double* __restrict__ o0, double* __restrict__ o1, double* __restrict__ o2, double* __restrict__ o3)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int b = inv_ptr[i], e = inv_ptr[i + 1];
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int k = b; k < e; ++k) {
        const long long g = inv_list[k];
        a0 += __ldcg(part + g);
        if (nq == 4) { a1 += __ldcg(part + part_stride + g); a2 += __ldcg(part + 2 * part_stride + g); a3 += __ldcg(part + 3 * part_stride + g); }
    }
    o0[i] = a0;
    if (nq == 4) { o1[i] = a1; o2[i] = a2; o3[i] = a3; }
}

size_t smem_bytes(bool field)
{
    return NTAB * sizeof(double) + CW * (field ? sizeof(WarpSmem<STRIDE_FLD>) : sizeof(WarpSmem<STRIDE_PSI>));
}

ColGeom geom_of(const pce_ctx* c, const Bins& b)
{
    ColGeom g;
    g.nbx = b.nc[0]; g.nby = b.nc[1]; g.nbz = b.nc[2]; g.Nz = c->wk.Ng[2]; g.P = c->wk.P;
    g.chunk = b.col_chunk;
    return g;
}

}  // namespace

// the cached-list kernels need bricks aligned with the periodic mesh and a support that meets a brick in one run
bool wave_cols_supported(const pce_ctx* c)
{
    for (int d = 0; d < 3; ++d)
        if (c->wk.Ng[d] % BR != 0 || c->wk.Ng[d] - c->wk.P < BR) return false;
    const char* e = getenv("PCE_NO_COLS");
    return !(e && e[0] == '1');
}

int wave_cols_init(pce_ctx* c)
{
    PCE_CUDA(c, cudaFuncSetAttribute(k_spread_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(false)));
    PCE_CUDA(c, cudaFuncSetAttribute(k_gather_cols<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(false)));
    PCE_CUDA(c, cudaFuncSetAttribute(k_gather_cols<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(true)));
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_cspread, k_spread_cols, CW * 32, smem_bytes(false)));
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_cgather, k_gather_cols<false>, CW * 32, smem_bytes(false)));
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_cgather_f, k_gather_cols<true>, CW * 32, smem_bytes(true)));
    if (c->occ_cspread < 1 || c->occ_cgather < 1 || c->occ_cgather_f < 1) { c->err = "column kernels do not fit on this device"; return PCE_ECUDA; }
    return PCE_OK;
}

// per mesh binning: records, key offsets, entries, work items (sizes are upper bounds: no host round trip per build)
int wave_cols_alloc(pce_ctx* c, Bins& b)
{
    const size_t n = (size_t)(b.n > 0 ? b.n : 1);
    const int span = (c->wk.P + 6) / BR + 1;  // bricks a support can meet per dimension
    const size_t nkeys = (size_t)b.nc[0] * b.nc[1] * c->wk.Ng[2];
    const size_t nbrick = (size_t)b.ncell;
    // crowded bricks are split only where there are too few bricks to fill the device (small meshes)
    b.col_chunk = (nbrick <= 4096) ? 64 : 0;
    b.col_ent_cap = (long long)n * span * span;
    const long long hits_cap = b.col_ent_cap * span;
    b.col_item_cap = (long long)nbrick + (b.col_chunk ? hits_cap / b.col_chunk + 1 : 0);
    PCE_CUDA(c, cudaMalloc(&b.hrec, n * sizeof(HitRec)));
    PCE_CUDA(c, cudaMalloc(&b.wu0, n * sizeof(double4)));
    PCE_CUDA(c, cudaMalloc(&b.col_cnt, (nkeys + 1) * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.col_start, (nkeys + 1) * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.col_ent, (size_t)b.col_ent_cap * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.item_start, (nbrick + 1) * sizeof(int)));
    c->bytes += (long long)(n * (sizeof(HitRec) + sizeof(double4)) + 2 * (nkeys + 1) * 4 + b.col_ent_cap * 4 + (nbrick + 1) * 4);
    if (b.col_chunk) {
        PCE_CUDA(c, cudaMalloc(&b.items, (size_t)b.col_item_cap * sizeof(int2)));
        PCE_CUDA(c, cudaMalloc(&b.col_scratch, (size_t)b.col_item_cap * 512 * sizeof(double)));
        PCE_CUDA(c, cudaMalloc(&b.col_arrive, nbrick * sizeof(int)));
        PCE_CUDA(c, cudaMemsetAsync(b.col_arrive, 0, nbrick * sizeof(int), c->st));
        c->bytes += (long long)(b.col_item_cap * (8 + 4096) + nbrick * 4);
    }
    if (c->p.flags & PCE_FLAG_DETERMINISTIC) {
        PCE_CUDA(c, cudaMalloc(&b.pair_start, (nbrick + 1) * sizeof(int)));
        PCE_CUDA(c, cudaMalloc(&b.inv_ptr, (n + 1) * sizeof(int)));
        c->bytes += (long long)((nbrick + 1 + n + 1) * 4);
    }
    b.nkeys = (long long)nkeys;
    b.qs_cols = reinterpret_cast<double*>(b.hrec) + (HITREC_Q_STRIDE - 1);  // the charge sits in the last 8 bytes of every record
    return PCE_OK;
}

void wave_cols_free(Bins& b)
{
    cudaFree(b.hrec); cudaFree(b.wu0); cudaFree(b.col_cnt); cudaFree(b.col_start); cudaFree(b.col_ent); cudaFree(b.item_start);
    cudaFree(b.items); cudaFree(b.col_scratch); cudaFree(b.col_arrive);
    cudaFree(b.pair_start); cudaFree(b.inv_ptr); cudaFree(b.inv_list);
}

// after bins_build: records and column lists of the binning's particles
int wave_cols_build(pce_ctx* c, Bins& b)
{
    if (b.n == 0) return PCE_OK;  // spread writes a zero mesh, gather has no targets
    const ColGeom g = geom_of(c, b);
    const int n = b.n, nkeys = (int)b.nkeys;
    k_hit_records<<<cdiv(n, 256), 256, 0, c->st>>>(n, c->wk, b.xs, b.ys, b.zs, b.hrec, b.wu0);
    PCE_CUDA(c, cudaMemsetAsync(b.col_cnt, 0, ((size_t)nkeys + 1) * sizeof(int), c->st));
    k_col_keys<false><<<cdiv(n, 256), 256, 0, c->st>>>(n, g, b.hrec, b.col_cnt, nullptr, nullptr);
    PCE_CUDA(c, cudaMemcpyAsync(b.col_start, b.col_cnt, ((size_t)nkeys + 1) * sizeof(int), cudaMemcpyDeviceToDevice, c->st));
    c->launches += 2;
    int rc = exclusive_scan(c, b.col_start, nkeys + 1);
    if (rc) return rc;
    PCE_CUDA(c, cudaMemsetAsync(b.col_cnt, 0, ((size_t)nkeys + 1) * sizeof(int), c->st));
    k_col_keys<true><<<cdiv(n, 256), 256, 0, c->st>>>(n, g, b.hrec, b.col_cnt, b.col_start, b.col_ent);
    // the fill counters are spent: the array now holds the list of keys with more than 8 entries (count at [nkeys], still 0)
    k_col_sort_small<<<cdiv(nkeys, 256), 256, 0, c->st>>>(nkeys, b.col_start, b.col_ent, b.col_cnt);
    k_col_sort_big<<<c->num_sm * 4, 128, 0, c->st>>>(nkeys, b.col_start, b.col_ent, b.col_cnt);
    c->launches += 3;
    b.n_items = b.ncell;
    if (b.col_chunk) {  // work items (brick, chunk): count, scan, fill; the total stays on the device side of the scan
        k_item_count<<<cdiv(b.ncell + 1, 256), 256, 0, c->st>>>(b.ncell, g, b.col_start, b.item_start);
        c->launches++;
        if ((rc = exclusive_scan(c, b.item_start, b.ncell + 1))) return rc;
        k_item_fill<<<cdiv(b.ncell, 256), 256, 0, c->st>>>(b.ncell, b.item_start, b.items);
        c->launches++;
        b.n_items = (int)b.col_item_cap;  // upper bound (sizes the launch); the kernels read the count from item_start[ncell]
    }
    if (c->p.flags & PCE_FLAG_DETERMINISTIC) {  // pair numbering and the per-particle pair lists of the deterministic gather
        k_pair_count<<<cdiv(b.ncell + 1, 256), 256, 0, c->st>>>(b.ncell, g, b.col_start, b.pair_start);
        k_inv_count<<<cdiv(n + 1, 256), 256, 0, c->st>>>(n, g.P, b.hrec, b.inv_ptr);
        c->launches += 2;
        if ((rc = exclusive_scan(c, b.pair_start, b.ncell + 1))) return rc;
        if ((rc = exclusive_scan(c, b.inv_ptr, n + 1))) return rc;
        int totals[2] = {0, 0};
        PCE_CUDA(c, cudaMemcpyAsync(&totals[0], b.pair_start + b.ncell, sizeof(int), cudaMemcpyDeviceToHost, c->st));
        PCE_CUDA(c, cudaMemcpyAsync(&totals[1], b.inv_ptr + n, sizeof(int), cudaMemcpyDeviceToHost, c->st));
        PCE_CUDA(c, cudaStreamSynchronize(c->st));
        if (totals[0] != totals[1] || totals[0] < 0) { c->err = "deterministic gather: pair lists inconsistent (or more than 2^31 pairs)"; return PCE_EINVAL; }
        b.n_pairs = totals[0];
        if (b.n_pairs > b.inv_cap) {
            cudaFree(b.inv_list);
            b.inv_list = nullptr;
            b.inv_cap = (long long)(b.n_pairs * 1.1) + 1024;
            PCE_CUDA(c, cudaMalloc(&b.inv_list, (size_t)b.inv_cap * sizeof(int)));
        }
        k_inv_fill<<<cdiv((long long)b.ncell * 32, 256), 256, 0, c->st>>>(b.ncell, g, b.col_start, b.col_ent, b.hrec, b.pair_start, b.inv_ptr, b.inv_list);
        c->launches++;
    }
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

static int grid_for(const pce_ctx* c, int per_sm, long long n_items)
{
    const long long want = (long long)c->num_sm * per_sm, need = (n_items + CW - 1) / CW;
    return (int)(want < need ? (want > 0 ? want : 1) : (need > 0 ? need : 1));
}

int wave_spread_cols(pce_ctx* c, const Bins& b)
{
    PassTimer t(c, PASS_SPREAD);
    if (b.n == 0) {  // no sources: the mesh is zero
        PCE_CUDA(c, cudaMemsetAsync(c->grid, 0, (size_t)c->wk.Ng[0] * c->wk.Ng[1] * c->wk.Ng[2] * sizeof(double), c->st));
        return PCE_OK;
    }
    PCE_CUDA(c, cudaMemsetAsync(c->work_ctr, 0, sizeof(int), c->st));
    k_spread_cols<<<grid_for(c, c->occ_cspread, b.n_items), CW * 32, smem_bytes(false), c->st>>>(
        c->wk, geom_of(c, b), b.col_start, b.col_ent, b.col_chunk ? b.items : nullptr, b.n_items, b.item_start, b.hrec, c->grid, b.col_scratch,
        b.col_arrive, c->work_ctr, c->skip_flag);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

int wave_gather_cols(pce_ctx* c, const Bins& b, bool field, double* psi_s, double* ex_s, double* ey_s, double* ez_s)
{
    if (b.n == 0) return PCE_OK;
    PassTimer t(c, PASS_GATHER);
    PCE_CUDA(c, cudaMemsetAsync(c->work_ctr, 0, sizeof(int), c->st));
    const bool det = (c->p.flags & PCE_FLAG_DETERMINISTIC) != 0;
    const int nq = field ? 4 : 1;
    const int* pair_start = nullptr;
    if (det) {  // partial sums per (brick, hit) pair and quantity
        const long long need = (long long)b.n_pairs * nq;
        if (need > c->part_cap) {
            krylov_invalidate_graph(c);  // the captured iteration names the old buffer
            cudaFree(c->gather_part);
            c->gather_part = nullptr;
            c->bytes -= c->part_cap * 8;
            c->part_cap = need + need / 8 + 1024;
            if (cudaMalloc(&c->gather_part, (size_t)c->part_cap * sizeof(double)) != cudaSuccess) { c->part_cap = 0; c->err = "out of device memory (gather partials)"; return PCE_ENOMEM; }
            c->bytes += c->part_cap * 8;
        }
        pair_start = b.pair_start;
    } else {
        PCE_CUDA(c, cudaMemsetAsync(psi_s, 0, (size_t)b.n * sizeof(double), c->st));
        if (field) {
            PCE_CUDA(c, cudaMemsetAsync(ex_s, 0, (size_t)b.n * sizeof(double), c->st));
            PCE_CUDA(c, cudaMemsetAsync(ey_s, 0, (size_t)b.n * sizeof(double), c->st));
            PCE_CUDA(c, cudaMemsetAsync(ez_s, 0, (size_t)b.n * sizeof(double), c->st));
        }
    }
    const int2* items = b.col_chunk ? b.items : nullptr;
    if (field) {
        k_gather_cols<true><<<grid_for(c, c->occ_cgather_f, b.n_items), CW * 32, smem_bytes(true), c->st>>>(
            c->wk, geom_of(c, b), b.col_start, b.col_ent, items, b.n_items, b.item_start, b.hrec, b.wu0, c->grid, psi_s, ex_s, ey_s, ez_s, c->work_ctr,
            c->skip_flag, pair_start, c->gather_part, (long long)b.n_pairs);
    } else {
        k_gather_cols<false><<<grid_for(c, c->occ_cgather, b.n_items), CW * 32, smem_bytes(false), c->st>>>(
            c->wk, geom_of(c, b), b.col_start, b.col_ent, items, b.n_items, b.item_start, b.hrec, b.wu0, c->grid, psi_s, nullptr, nullptr, nullptr, c->work_ctr,
            c->skip_flag, pair_start, c->gather_part, (long long)b.n_pairs);
    }
    c->launches++;
    if (det) {
        k_gather_finish<<<cdiv(b.n, 256), 256, 0, c->st>>>(b.n, nq, b.inv_ptr, b.inv_list, c->gather_part, (long long)b.n_pairs, psi_s, ex_s, ey_s, ez_s);
        c->launches++;
    }
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
