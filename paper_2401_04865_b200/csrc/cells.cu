// cells.cu -- linked-cell binning by counting sort ("linear
// complexity linked cell algorithm"), SoA reorder, and the integer scan it needs.
// Deterministic: the order inside a cell is the caller's index order.
#include "pce_internal.h"

// ---------------------------------------------------------------- exclusive scan (int32)
constexpr int SCAN_T = 256, SCAN_E = 8, SCAN_B = SCAN_T * SCAN_E;

__global__ void k_scan_local(int* data, int* bsum, int n)
{
    __shared__ int sh[SCAN_T];
    const int tid = threadIdx.x;
    const long long base = (long long)blockIdx.x * SCAN_B + (long long)tid * SCAN_E;
    int v[SCAN_E], s = 0;
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        long long i = base + e;
        v[e] = (i < n) ? data[i] : 0;
        s += v[e];
    }
    sh[tid] = s;
    __syncthreads();
    for (int off = 1; off < SCAN_T; off <<= 1) {
        int t = (tid >= off) ? sh[tid - off] : 0;
        __syncthreads();
        sh[tid] += t;
        __syncthreads();
    }
    int run = sh[tid] - s;
    if (tid == SCAN_T - 1) bsum[blockIdx.x] = sh[tid];
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        long long i = base + e;
        if (i < n) data[i] = run;
        run += v[e];
    }
}

__global__ void k_scan_bsum(int* bsum, int nb)
{
    __shared__ int sh[1024];
    __shared__ int carry;
    const int tid = threadIdx.x;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + tid;
        const int v = (i < nb) ? bsum[i] : 0;
        sh[tid] = v;
        __syncthreads();
        for (int off = 1; off < 1024; off <<= 1) {
            int t = (tid >= off) ? sh[tid - off] : 0;
            __syncthreads();
            sh[tid] += t;
            __syncthreads();
        }
        const int incl = sh[tid];
        const int c0 = carry;
        __syncthreads();
        if (i < nb) bsum[i] = c0 + incl - v;
        if (tid == 1023) carry = c0 + incl;
        __syncthreads();
    }
}

__global__ void k_scan_add(int* data, const int* bsum, int n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) data[i] += bsum[i / SCAN_B];
}

int exclusive_scan(pce_ctx* c, int* data, int n)
{
    const int nb = cdiv(n, SCAN_B);
    if ((size_t)nb > c->scan_tmp_n) {
        if (c->scan_tmp) cudaFree(c->scan_tmp);
        c->scan_tmp_n = (size_t)nb * 2 + 64;
        PCE_CUDA(c, cudaMalloc(&c->scan_tmp, c->scan_tmp_n * sizeof(int)));
    }
    k_scan_local<<<nb, SCAN_T, 0, c->st>>>(data, c->scan_tmp, n);
    k_scan_bsum<<<1, 1024, 0, c->st>>>(c->scan_tmp, nb);
    k_scan_add<<<cdiv(n, 256), 256, 0, c->st>>>(data, c->scan_tmp, n);
    c->launches += 3;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// ---------------------------------------------------------------- positions
__global__ void k_wrap(int n, const double* __restrict__ xi, const double* __restrict__ yi, const double* __restrict__ zi,
                       double* __restrict__ xo, double* __restrict__ yo, double* __restrict__ zo, double Lx, double Ly, double Lz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x = xi[i], y = yi[i], z = zi[i];
    x -= Lx * floor(x / Lx);
    y -= Ly * floor(y / Ly);
    z -= Lz * floor(z / Lz);
    if (x >= Lx) x = 0.0;
    if (y >= Ly) y = 0.0;
    if (z >= Lz) z = 0.0;
    xo[i] = x; yo[i] = y; zo[i] = z;
}

int wrap_positions(pce_ctx* c, int n, const double* xi, const double* yi, const double* zi, double* xo, double* yo, double* zo)
{
    if (n == 0) return PCE_OK;
    k_wrap<<<cdiv(n, 256), 256, 0, c->st>>>(n, xi, yi, zi, xo, yo, zo, c->p.L[0], c->p.L[1], c->p.L[2]);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

__global__ void k_gather_perm(int n, const int* __restrict__ perm, const double* __restrict__ in, double* __restrict__ out, int stride)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[(size_t)i * stride] = in[perm[i]];
}

// out[i * out_stride] = in[perm[i]] (stride HITREC_Q_STRIDE = 8: the charge slot of the 64-byte hit records, wave_cols.cu)
int gather_by_perm(pce_ctx* c, int n, const int* perm, const double* in, double* out, int out_stride)
{
    if (n == 0) return PCE_OK;
    k_gather_perm<<<cdiv(n, 256), 256, 0, c->st>>>(n, perm, in, out, out_stride);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

// ---------------------------------------------------------------- binning
__global__ void k_cell_count(int n, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                             int ncx, int ncy, int ncz, double sx, double sy, double sz, int mx, int my, int mz, int dvx, int dvy,
                             int dvz, int shx, int shy, int shz, int* __restrict__ cell_of, int* __restrict__ count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    // index along each dimension, cyclically shifted by sh (mesh bins only), then divided into bins
    int ix = min((int)(x[i] * sx), mx) + shx, iy = min((int)(y[i] * sy), my) + shy, iz = min((int)(z[i] * sz), mz) + shz;
    if (ix > mx) ix -= mx + 1;
    if (iy > my) iy -= my + 1;
    if (iz > mz) iz -= mz + 1;
    int cx = min(ix / dvx, ncx - 1);
    int cy = min(iy / dvy, ncy - 1);
    int cz = min(iz / dvz, ncz - 1);
    const int cidx = (cz * ncy + cy) * ncx + cx;
    cell_of[i] = cidx;
    atomicAdd(&count[cidx], 1);
}

__global__ void k_cell_scatter(int n, const int* __restrict__ cell_of, const int* __restrict__ cell_start, int* __restrict__ fill,
                               int* __restrict__ perm)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int cidx = cell_of[i];
    const int slot = atomicAdd(&fill[cidx], 1);
    perm[cell_start[cidx] + slot] = i;
}

// order every cell's entries by caller index (rank by counting): one thread per sorted slot, so that a crowded cell -- a
// 2562-bead sphere inside a few cells -- is shared by as many threads as it has entries (one warp per cell took n_cell^2 / 32 steps)
__global__ void __launch_bounds__(256)
k_cell_rank(int n, const int* __restrict__ cell_of, const int* __restrict__ cell_start, const int* __restrict__ perm_in,
            int* __restrict__ perm_out)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int mine = perm_in[s];
    const int cidx = cell_of[mine];
    const int b = cell_start[cidx], e = cell_start[cidx + 1];
    int rank = 0;
    for (int j = b; j < e; ++j) rank += (__ldg(perm_in + j) < mine);
    perm_out[b + rank] = mine;
}

__global__ void k_iota(int n, int* p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = i;
}

__global__ void k_gather3(int n, const int* __restrict__ perm, const double* __restrict__ x, const double* __restrict__ y,
                          const double* __restrict__ z, double* __restrict__ xs, double* __restrict__ ys, double* __restrict__ zs,
                          int* __restrict__ inv)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int j = perm[i];
    inv[j] = i;
    xs[i] = x[j]; ys[i] = y[j]; zs[i] = z[j];
}

// out[cell] = number of 32-target chunks of the cell, out[ncell] = 0 (then scanned in place)
__global__ void k_chunk_count(int ncell, const int* __restrict__ cell_start, int* __restrict__ out)
{
    const int cidx = blockIdx.x * blockDim.x + threadIdx.x;
    if (cidx > ncell) return;
    out[cidx] = (cidx < ncell) ? (cell_start[cidx + 1] - cell_start[cidx] + 31) / 32 : 0;
}

int bins_alloc(pce_ctx* c, Bins& b, int n, const int nc[3], const int range[3])
{
    bins_free(b);
    b.n = n;
    for (int d = 0; d < 3; ++d) {
        b.nc[d] = nc[d]; b.range[d] = range[d]; b.L[d] = c->p.L[d];
        b.scale[d] = nc[d] / c->p.L[d]; b.imax[d] = nc[d] - 1; b.div[d] = 1;
    }
    b.ncell = nc[0] * nc[1] * nc[2];
    const size_t ni = (size_t)(n > 0 ? n : 1);
    PCE_CUDA(c, cudaMalloc(&b.cell_of, ni * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.cell_start, ((size_t)b.ncell + 1) * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.cell_fill, ((size_t)b.ncell + 1) * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.perm, ni * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.perm_tmp, ni * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.inv, ni * sizeof(int)));
    PCE_CUDA(c, cudaMalloc(&b.xs, ni * sizeof(double)));
    PCE_CUDA(c, cudaMalloc(&b.ys, ni * sizeof(double)));
    PCE_CUDA(c, cudaMalloc(&b.zs, ni * sizeof(double)));
    PCE_CUDA(c, cudaMalloc(&b.qs, ni * sizeof(double)));
    c->bytes += (long long)(ni * (4 * 4 + 4 * 8) + ((size_t)b.ncell + 1) * 8);
    return PCE_OK;
}

// real-space binnings also carry the chunk list of the direct pass
int bins_alloc_chunks(pce_ctx* c, Bins& b)
{
    PCE_CUDA(c, cudaMalloc(&b.chunk_start, ((size_t)b.ncell + 1) * sizeof(int)));
    c->bytes += (long long)(((size_t)b.ncell + 1) * 4);
    return PCE_OK;
}

int bins_alloc_tiles(pce_ctx* c, Bins& b, int n, int tile)
{
    int nc[3], range[3] = {1, 1, 1};
    for (int d = 0; d < 3; ++d) nc[d] = (c->p.Ng[d] + tile - 1) / tile;
    int rc = bins_alloc(c, b, n, nc, range);
    if (rc) return rc;
    // the same 1/h the mesh kernels use, so that floor(x/h) agrees bit for bit
    // bins are shifted by P/2 mod tile so that the mesh cells whose support meets a brick span the fewest bins
    for (int d = 0; d < 3; ++d) {
        b.scale[d] = c->wk.inv_h[d]; b.imax[d] = c->p.Ng[d] - 1; b.div[d] = tile; b.shift[d] = (c->wk.P / 2) % tile;  // the active window (wave_select)
    }
    return PCE_OK;
}

void bins_free(Bins& b)
{
    cudaFree(b.cell_of); cudaFree(b.cell_start); cudaFree(b.cell_fill); cudaFree(b.perm); cudaFree(b.perm_tmp); cudaFree(b.inv);
    cudaFree(b.xs); cudaFree(b.ys); cudaFree(b.zs); cudaFree(b.qs);
    cudaFree(b.ws0); cudaFree(b.wcf); cudaFree(b.chunk_start);
    wave_cols_free(b);
    b = Bins();
}

// x, y, z: wrapped positions of the subset (first b.n entries)
int bins_build(pce_ctx* c, Bins& b, const double* x, const double* y, const double* z)
{
    const int n = b.n;
    if (n == 0) {
        PCE_CUDA(c, cudaMemsetAsync(b.cell_start, 0, ((size_t)b.ncell + 1) * sizeof(int), c->st));
        return PCE_OK;
    }
    if (b.ncell == 1) {
        const int hs[2] = {0, n};
        PCE_CUDA(c, cudaMemcpyAsync(b.cell_start, hs, 2 * sizeof(int), cudaMemcpyHostToDevice, c->st));
        PCE_CUDA(c, cudaMemsetAsync(b.cell_of, 0, (size_t)n * sizeof(int), c->st));
        k_iota<<<cdiv(n, 256), 256, 0, c->st>>>(n, b.perm);
        c->launches++;
    } else {
        PCE_CUDA(c, cudaMemsetAsync(b.cell_start, 0, ((size_t)b.ncell + 1) * sizeof(int), c->st));
        PCE_CUDA(c, cudaMemsetAsync(b.cell_fill, 0, ((size_t)b.ncell + 1) * sizeof(int), c->st));
        k_cell_count<<<cdiv(n, 256), 256, 0, c->st>>>(n, x, y, z, b.nc[0], b.nc[1], b.nc[2], b.scale[0], b.scale[1], b.scale[2],
                                                      b.imax[0], b.imax[1], b.imax[2], b.div[0], b.div[1], b.div[2], b.shift[0],
                                                      b.shift[1], b.shift[2], b.cell_of,
                                                      b.cell_start);
        c->launches++;
        int rc = exclusive_scan(c, b.cell_start, b.ncell + 1);
        if (rc) return rc;
        k_cell_scatter<<<cdiv(n, 256), 256, 0, c->st>>>(n, b.cell_of, b.cell_start, b.cell_fill, b.perm_tmp);
        k_cell_rank<<<cdiv(n, 256), 256, 0, c->st>>>(n, b.cell_of, b.cell_start, b.perm_tmp, b.perm);
        c->launches += 2;
    }
    k_gather3<<<cdiv(n, 256), 256, 0, c->st>>>(n, b.perm, x, y, z, b.xs, b.ys, b.zs, b.inv);
    c->launches++;
    if (b.chunk_start) {  // real-space binnings: work items of the direct pass = (cell, chunk of 32 targets)
        k_chunk_count<<<cdiv(b.ncell + 1, 256), 256, 0, c->st>>>(b.ncell, b.cell_start, b.chunk_start);
        c->launches++;
        int rc = exclusive_scan(c, b.chunk_start, b.ncell + 1);
        if (rc) return rc;
    }
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
