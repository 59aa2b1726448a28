// precond.cu -- block-Jacobi preconditioner of the induced-charge Krylov solve (eq. 13, PAPER.md:131;
// SURVEY.md 8(f) f1).  The paper solves eq. 13 "iteratively" without naming a preconditioner;
// the solution is unique (M is SPD), so a preconditioner changes the iteration count only.
//
// For every rigid body i with n_i <= PC_MAX_BODY beads the FREE-SPACE potential tensor of its own beads,
//     A_jk = M(|r_ij - r_ik|)  with eq. 10 (reading G1),  A_jj = 1/(4 pi eps a),
// depends on the body-frame bead positions r_ij only, i.e. it is invariant under the rigid motion of the body
// (PAPER.md:107-111): it is built and inverted ONCE per pce_set_system and reused by every later solve.
//   B_i = A^-1 - u u^T / (1^T u),  u = A^-1 1
// is the inverse of A on the zero-net-charge subspace of the body (the constraint sum_j q_ij = Q_i of eq. 11),
// symmetric positive semi-definite with null vector 1.  The Krylov driver applies z = P B r (P = remove the
// per-body mean) as one dense matrix-vector product per body.  B is stored in bf16 for large systems (it only steers the
// search directions; every quantity that enters the result -- residual, step lengths, charges -- stays fp64;
// measured: 30 iterations at config 5 with fp32, with 11 and with 8 mantissa bits alike), which quarters the HBM
// bytes of the apply: sum_i 2 n_i^2 bytes per iteration (1 GB at 500 x 1000 beads).  Rows are padded to a multiple
// of 8 entries (16-byte loads), rounding is to nearest even and symmetric (B_jk and B_kj round alike).
//
// Inversion: in-place block Gauss-Jordan without pivoting (every pivot block is a Schur complement of an SPD
// matrix), 32 pivots per step.  Per step a panel kernel (reads A only; writes D^-1, the row panel D^-1 A_K:,
// the old column panel A_:K and -A_:K D^-1) and an update kernel (64x64 tiles, 4x4 per thread; the only
// writer of A) run over all bodies of a chunk at once.
#include "pce_internal.h"

#include <cstdlib>

constexpr int GJB = 32;            // pivots per block step
__host__ __device__ constexpr int pc_ld(int n) { return (n + 7) & ~7; }  // row stride of the stored block (16-byte loads)
constexpr int PC_MAX_BODY = 4096;  // larger bodies are left unpreconditioned (scaled identity)
constexpr long long PC_CHUNK_ELEMS = 1ll << 28;  // fp64 work matrix per chunk of bodies: 2 GB
constexpr long long PC_MAX_ELEMS = 3ll << 30;    // total bf16 storage cap: 6 GB

struct PcBody {          // one preconditioned body inside the current chunk
    int j0, n;           // first bead, bead count
    int body, pad;       // body index
    long long woff;      // offset of its n x n fp64 work matrix
    long long poff;      // offset of its panels (3 x n x GJB + GJB x GJB doubles)
    long long boff;      // offset (entries) of its matrix (row stride pc_ld(n)) in pc_B
};

// ---------------------------------------------------------------- A_jk = M_free(|r_j - r_k|), eq. 10
__global__ void __launch_bounds__(256)
k_pc_fill(const PcBody* __restrict__ bodies, const double* __restrict__ rx, const double* __restrict__ ry, const double* __restrict__ rz,
          double a, double inv_eps, double* __restrict__ work)
{
    const PcBody B = bodies[blockIdx.z];
    const int j = blockIdx.x * 16 + (threadIdx.x & 15), i = blockIdx.y * 16 + (threadIdx.x >> 4);
    if (i >= B.n || j >= B.n) return;
    const double dx = rx[B.j0 + i] - rx[B.j0 + j], dy = ry[B.j0 + i] - ry[B.j0 + j], dz = rz[B.j0 + i] - rz[B.j0 + j];
    const double r = sqrt(dx * dx + dy * dy + dz * dz);
    const double inv4pi = 1.0 / (4.0 * PCE_PI);
    const double v = (r >= 2.0 * a) ? inv4pi / r : inv4pi * (4.0 * a - r) / (4.0 * a * a);  // M(0) = 1/(4 pi a)
    work[B.woff + (long long)i * B.n + j] = v * inv_eps;
}

// ---------------------------------------------------------------- block Gauss-Jordan, panel kernel
// grid (ceil(nmax/256), bodies).  Every CTA inverts the pivot block D = A_KK (redundantly, 32^3 work) and
// produces, for its 256 columns / rows:  Rw = D^-1 A_K,:  (GJB x n),  Cl = A_:,K (n x GJB),  Cn = -A_:,K D^-1.
__global__ void __launch_bounds__(256)
k_pc_panel(const PcBody* __restrict__ bodies, int step, const double* __restrict__ work, double* __restrict__ panels)
{
    __shared__ double D[GJB][GJB + 1];
    __shared__ double colp[GJB];
    const PcBody B = bodies[blockIdx.y];
    const int n = B.n, k0 = step * GJB;
    if (k0 >= n || (int)blockIdx.x * 256 >= n) return;
    const int kb = min(GJB, n - k0);
    const double* A = work + B.woff;
    const int tid = threadIdx.x;
    for (int e = tid; e < GJB * GJB; e += 256) {
        const int i = e / GJB, j = e % GJB;
        D[i][j] = (i < kb && j < kb) ? A[(long long)(k0 + i) * n + k0 + j] : (i == j ? 1.0 : 0.0);
    }
    __syncthreads();
    for (int p = 0; p < kb; ++p) {
        const double piv = 1.0 / D[p][p];
        if (tid < GJB) colp[tid] = D[tid][p];
        __syncthreads();
        if (tid < GJB) D[p][tid] = (tid == p) ? piv : D[p][tid] * piv;
        __syncthreads();
        for (int e = tid; e < GJB * GJB; e += 256) {
            const int i = e / GJB, j = e % GJB;
            if (i != p) D[i][j] = (j == p) ? -colp[i] * piv : D[i][j] - colp[i] * D[p][j];
        }
        __syncthreads();
    }
    double* Rw = panels + B.poff;                       // [GJB][n]
    double* Cl = Rw + (long long)GJB * n;               // [n][GJB]
    double* Cn = Cl + (long long)GJB * n;               // [n][GJB]
    double* Di = Cn + (long long)GJB * n;               // [GJB][GJB]
    if (blockIdx.x == 0)
        for (int e = tid; e < GJB * GJB; e += 256) Di[e] = D[e / GJB][e % GJB];
    const int c = blockIdx.x * 256 + tid;  // column of the row panel and row of the column panel
    if (c >= n) return;
    double v[GJB];
#pragma unroll
    for (int m = 0; m < GJB; ++m) v[m] = (m < kb) ? A[(long long)(k0 + m) * n + c] : 0.0;
#pragma unroll 4
    for (int k = 0; k < GJB; ++k) {
        double s = 0.0;
#pragma unroll
        for (int m = 0; m < GJB; ++m) s = fma(D[k][m], v[m], s);
        Rw[(long long)k * n + c] = s;
    }
#pragma unroll
    for (int m = 0; m < GJB; ++m) v[m] = (m < kb) ? A[(long long)c * n + k0 + m] : 0.0;
#pragma unroll
    for (int m = 0; m < GJB; ++m) Cl[(long long)c * GJB + m] = v[m];
#pragma unroll 4
    for (int k = 0; k < GJB; ++k) {
        double s = 0.0;
#pragma unroll
        for (int m = 0; m < GJB; ++m) s = fma(v[m], D[m][k], s);
        Cn[(long long)c * GJB + k] = -s;
    }
}

// ---------------------------------------------------------------- block Gauss-Jordan, update kernel (only writer of A)
// grid (ceil(nmax/64), ceil(nmax/64), bodies), 256 threads, 4x4 entries per thread:
//   i, j outside K: A_ij -= Cl_i . Rw_j ;  i in K: A_ij = Rw_ij ;  j in K: A_ij = Cn_ij ;  both: D^-1
__global__ void __launch_bounds__(256)
k_pc_update(const PcBody* __restrict__ bodies, int step, double* __restrict__ work, const double* __restrict__ panels)
{
    __shared__ double sC[64][GJB + 1];
    __shared__ double sR[GJB][64 + 2];
    const PcBody B = bodies[blockIdx.z];
    const int n = B.n, k0 = step * GJB;
    const int i0 = blockIdx.y * 64, j0 = blockIdx.x * 64;
    if (k0 >= n || i0 >= n || j0 >= n) return;
    double* A = work + B.woff;
    const double* Rw = panels + B.poff;
    const double* Cl = Rw + (long long)GJB * n;
    const double* Cn = Cl + (long long)GJB * n;
    const double* Di = Cn + (long long)GJB * n;
    const int tid = threadIdx.x;
    for (int e = tid; e < 64 * GJB; e += 256) {
        const int r = e / GJB, m = e % GJB;
        sC[r][m] = (i0 + r < n) ? Cl[(long long)(i0 + r) * GJB + m] : 0.0;
    }
    for (int e = tid; e < GJB * 64; e += 256) {
        const int m = e / 64, cc = e % 64;
        sR[m][cc] = (j0 + cc < n) ? Rw[(long long)m * n + j0 + cc] : 0.0;
    }
    __syncthreads();
    const int tx = tid & 15, ty = tid >> 4;  // columns j0 + tx + 16 b, rows i0 + ty + 16 a
    double acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
#pragma unroll 8
    for (int m = 0; m < GJB; ++m) {
        double cv[4], rv[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) cv[a] = sC[ty + 16 * a][m];
#pragma unroll
        for (int b = 0; b < 4; ++b) rv[b] = sR[m][tx + 16 * b];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) acc[a][b] = fma(cv[a], rv[b], acc[a][b]);
    }
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const int i = i0 + ty + 16 * a;
        if (i >= n) continue;
        const bool ik = (i >= k0 && i < k0 + GJB);
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int j = j0 + tx + 16 * b;
            if (j >= n) continue;
            const bool jk = (j >= k0 && j < k0 + GJB);
            double* p = A + (long long)i * n + j;
            double v;
            if (ik && jk) v = Di[(i - k0) * GJB + (j - k0)];
            else if (ik) v = Rw[(long long)(i - k0) * n + j];
            else if (jk) v = Cn[(long long)i * GJB + (j - k0)];
            else v = *p - acc[a][b];
            *p = v;
        }
    }
}

// u_i = sum_j Ainv_ij (one warp per row), fixed order
__global__ void __launch_bounds__(256)
k_pc_rowsum(const PcBody* __restrict__ bodies, const double* __restrict__ work, double* __restrict__ u)
{
    const PcBody B = bodies[blockIdx.y];
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= B.n) return;
    const double* A = work + B.woff + (long long)row * B.n;
    double s = 0.0;
    for (int j = lane; j < B.n; j += 32) s += A[j];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if (lane == 0) u[B.j0 + row] = s;
}

// s_b = sum_i u_i (one CTA per body)
__global__ void __launch_bounds__(256)
k_pc_usum(const PcBody* __restrict__ bodies, const double* __restrict__ u, double* __restrict__ usum, double* __restrict__ inv_s_body)
{
    __shared__ double sh[8];
    const PcBody B = bodies[blockIdx.x];
    double s = 0.0;
    for (int j = threadIdx.x; j < B.n; j += 256) s += u[B.j0 + j];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; ++k) t += sh[k];
        usum[blockIdx.x] = t;
        inv_s_body[B.body] = 1.0 / t;  // kept: A^-1 r = B r + u (u.r)/s for the unconstrained solves (capacitance tensor)
    }
}

// B_ij = (Ainv_ij + Ainv_ji)/2 - u_i u_j / s   -> fp32 (32x32 tiles, transposed read through shared memory)
template <bool BF16>
__global__ void __launch_bounds__(256)
k_pc_final(const PcBody* __restrict__ bodies, const double* __restrict__ work, const double* __restrict__ u,
           const double* __restrict__ usum, void* __restrict__ Bout)
{
    __shared__ double tT[32][33];
    const PcBody B = bodies[blockIdx.z];
    const int n = B.n, i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
    if (i0 >= n || j0 >= n) return;
    const double* A = work + B.woff;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8)  // tile (j0.., i0..) of A, to be read transposed
        tT[r][tx] = (j0 + r < n && i0 + tx < n) ? A[(long long)(j0 + r) * n + i0 + tx] : 0.0;
    __syncthreads();
    const double inv_s = 1.0 / usum[blockIdx.z];
    for (int r = ty; r < 32; r += 8) {
        const int i = i0 + r, j = j0 + tx;
        if (i < n && j < n) {
            const double v = 0.5 * (A[(long long)i * n + j] + tT[tx][r]) - u[B.j0 + i] * u[B.j0 + j] * inv_s;
            const long long o = B.boff + (long long)i * pc_ld(n) + j;
            if (BF16) {
                const unsigned u32 = __float_as_uint((float)v);
                static_cast<unsigned short*>(Bout)[o] = (unsigned short)((u32 + 0x7fffu + ((u32 >> 16) & 1u)) >> 16);  // nearest even
            } else {
                static_cast<float*>(Bout)[o] = (float)v;
            }
        }
    }
}

// ---------------------------------------------------------------- apply: z_raw = B r (rows of one body per CTA)
struct PcRows { int j0, n, row0; int pad; long long boff; };  // CTA -> body, first row

constexpr int PC_ROWS = 64;  // rows per CTA (8 per warp: one shared-memory read of the residual serves 8 rows)

__device__ __forceinline__ double bf16_lo(unsigned w) { return (double)__uint_as_float(w << 16); }
__device__ __forceinline__ double bf16_hi(unsigned w) { return (double)__uint_as_float(w & 0xffff0000u); }

template <bool BF16>
__global__ void __launch_bounds__(256)
k_pc_apply(const PcRows* __restrict__ rows, const void* __restrict__ Bv, const double* __restrict__ r, double* __restrict__ z,
           const int* __restrict__ skip)
{
    if (skip && *skip) return;  // solver already converged (krylov.cu)
    extern __shared__ double sr[];  // the body's residual, zero-padded to the row stride
    const PcRows R = rows[blockIdx.x];
    const int ld = pc_ld(R.n);
    for (int j = threadIdx.x; j < ld; j += 256) sr[j] = (j < R.n) ? r[R.j0 + j] : 0.0;
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // the warp's 4 rows are swept together: one read of the residual from shared memory serves 4 rows, and 4 independent
    // 16-byte loads (8 entries each) are in flight per lane
    constexpr int NR = PC_ROWS / 8;
    constexpr int ES = BF16 ? 2 : 4;   // bytes per stored entry
    const unsigned char* Br[NR];
    bool live[NR];
    double acc[NR];
#pragma unroll
    for (int k = 0; k < NR; ++k) {
        const int row = R.row0 + warp + 8 * k;
        live[k] = row < R.n;
        Br[k] = static_cast<const unsigned char*>(Bv) + (R.boff + (long long)(live[k] ? row : 0) * ld) * ES;
        acc[k] = 0.0;
    }
    for (int j = 8 * lane; j < ld; j += 256) {
        const double2 r01 = *reinterpret_cast<const double2*>(sr + j), r23 = *reinterpret_cast<const double2*>(sr + j + 2);
        const double2 r45 = *reinterpret_cast<const double2*>(sr + j + 4), r67 = *reinterpret_cast<const double2*>(sr + j + 6);
#pragma unroll
        for (int k = 0; k < NR; ++k) {
            double a = acc[k];
            if (!BF16) {
                const float4 b0 = __ldg(reinterpret_cast<const float4*>(Br[k] + (size_t)j * 4)), b1 = __ldg(reinterpret_cast<const float4*>(Br[k] + (size_t)j * 4 + 16));
                a = fma((double)b0.x, r01.x, a); a = fma((double)b0.y, r01.y, a); a = fma((double)b0.z, r23.x, a); a = fma((double)b0.w, r23.y, a);
                a = fma((double)b1.x, r45.x, a); a = fma((double)b1.y, r45.y, a); a = fma((double)b1.z, r67.x, a); a = fma((double)b1.w, r67.y, a);
                acc[k] = a;
                continue;
            }
            const uint4 b = __ldg(reinterpret_cast<const uint4*>(Br[k] + (size_t)j * 2));
            a = fma(bf16_lo(b.x), r01.x, a); a = fma(bf16_hi(b.x), r01.y, a);
            a = fma(bf16_lo(b.y), r23.x, a); a = fma(bf16_hi(b.y), r23.y, a);
            a = fma(bf16_lo(b.z), r45.x, a); a = fma(bf16_hi(b.z), r45.y, a);
            a = fma(bf16_lo(b.w), r67.x, a); a = fma(bf16_hi(b.w), r67.y, a);
            acc[k] = a;
        }
    }
#pragma unroll
    for (int k = 0; k < NR; ++k) {
        double sum = acc[k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
        if (lane == 0 && live[k]) z[R.j0 + R.row0 + warp + 8 * k] = sum;
    }
}

// beads of bodies without a dense block: z = r / M(0) = 4 pi eps a r
__global__ void k_pc_identity(int n, const unsigned char* __restrict__ has_block, const int* __restrict__ body_of, double scale,
                              const double* __restrict__ r, double* __restrict__ z, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && !has_block[body_of[i]]) z[i] = scale * r[i];
}

// ---------------------------------------------------------------- host
void precond_free(pce_ctx* c)
{
    cudaFree(c->pc_B); cudaFree(c->pc_rows); cudaFree(c->pc_has); cudaFree(c->pc_u); cudaFree(c->pc_invs);
    c->pc_B = nullptr; c->pc_rows = nullptr; c->pc_has = nullptr; c->pc_u = nullptr; c->pc_invs = nullptr;
    c->pc_on = false; c->pc_nrows_cta = 0; c->pc_max_n = 0; c->pc_bytes = 0; c->pc_nblock = 0;
}

// Build B_i for every body (once per pce_set_system: needs rx, ry, rz of bodies_setup).
int precond_setup(pce_ctx* c)
{
    precond_free(c);
    if ((c->p.flags & PCE_FLAG_NO_PRECOND) || c->Nbody == 0 || c->Nbead == 0) return PCE_OK;
    const int nb = c->Nbody;
    const std::vector<int>& off = c->body_off_h;
    // which bodies get a dense block
    std::vector<unsigned char> has(nb, 0);
    std::vector<PcBody> all;
    long long total = 0;
    int max_n = 0;
    for (int b = 0; b < nb; ++b) {
        const int n = off[b + 1] - off[b];
        if (n < 2 || n > PC_MAX_BODY || total + (long long)n * n > PC_MAX_ELEMS) continue;
        PcBody B;
        B.j0 = off[b]; B.n = n; B.body = b; B.pad = 0; B.woff = 0; B.poff = 0; B.boff = total;
        total += (long long)n * pc_ld(n);  // rows padded to 8 entries: 16-byte aligned for the uint4 loads
        all.push_back(B);
        has[b] = 1;
        if (n > max_n) max_n = n;
    }
    if (all.empty()) return PCE_OK;
    // storage precision: bf16 where the apply is a real share of the iteration (many bodies, > 128 MB in fp32: the iteration
    // count is set by the coupling between bodies, 30 at config 5 either way), fp32 for few or small bodies, whose blocks are
    // nearly exact inverses of the whole operator (config 3: 3 iterations with fp32, 6 with bf16)
    c->pc_bf16 = (int)all.size() >= 16 && total * 4 > (128ll << 20);
    const size_t esize = c->pc_bf16 ? sizeof(unsigned short) : sizeof(float);
    if (cudaMalloc(&c->pc_B, (size_t)total * esize) != cudaSuccess) {
        cudaGetLastError();
        c->pc_B = nullptr;
        return PCE_OK;  // no room for the preconditioner: plain CG (the result does not depend on it)
    }
    PCE_CUDA(c, cudaMemsetAsync(c->pc_B, 0, (size_t)total * esize, c->st));  // the row padding must read as 0
    PCE_CUDA(c, cudaMalloc(&c->pc_has, (size_t)nb));
    PCE_CUDA(c, cudaMemcpyAsync(c->pc_has, has.data(), (size_t)nb, cudaMemcpyHostToDevice, c->st));
    // CTA -> (body, first row) map of the apply kernel
    std::vector<PcRows> rows;
    for (const PcBody& B : all)
        for (int r0 = 0; r0 < B.n; r0 += PC_ROWS) rows.push_back({B.j0, B.n, r0, 0, B.boff});
    PCE_CUDA(c, cudaMalloc(&c->pc_rows, rows.size() * sizeof(PcRows)));
    PCE_CUDA(c, cudaMemcpyAsync(c->pc_rows, rows.data(), rows.size() * sizeof(PcRows), cudaMemcpyHostToDevice, c->st));
    PCE_CUDA(c, cudaStreamSynchronize(c->st));
    c->pc_nrows_cta = (int)rows.size();
    c->pc_max_n = max_n;
    c->pc_nblock = (int)all.size();
    c->pc_bytes = total * (long long)esize;
    c->bytes += c->pc_bytes;
    if ((size_t)pc_ld(max_n) * sizeof(double) > 48 * 1024)
    {
        PCE_CUDA(c, cudaFuncSetAttribute(k_pc_apply<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(pc_ld(max_n) * sizeof(double))));
        PCE_CUDA(c, cudaFuncSetAttribute(k_pc_apply<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(pc_ld(max_n) * sizeof(double))));
    }

    // chunks of bodies whose fp64 work matrices fit PC_CHUNK_ELEMS
    double *work = nullptr, *panels = nullptr, *u = nullptr, *usum = nullptr;
    PcBody* dbod = nullptr;
    long long work_cap = 0, pan_cap = 0;
    int nb_cap = 0;
    int rc = PCE_OK;
    size_t i = 0;
    PCE_CUDA(c, cudaMalloc(&c->pc_u, (size_t)c->Nbead * sizeof(double)));
    PCE_CUDA(c, cudaMalloc(&c->pc_invs, (size_t)nb * sizeof(double)));
    PCE_CUDA(c, cudaMemsetAsync(c->pc_u, 0, (size_t)c->Nbead * sizeof(double), c->st));
    PCE_CUDA(c, cudaMemsetAsync(c->pc_invs, 0, (size_t)nb * sizeof(double), c->st));
    u = c->pc_u;  // u = A^-1 1 per body, kept
    while (i < all.size() && rc == PCE_OK) {
        std::vector<PcBody> ch;
        long long w = 0, pz = 0;
        int nmax = 0;
        while (i < all.size() && (ch.empty() || w + (long long)all[i].n * all[i].n <= PC_CHUNK_ELEMS)) {
            PcBody B = all[i++];
            B.woff = w; B.poff = pz;
            w += (long long)B.n * B.n;
            pz += 3ll * GJB * B.n + GJB * GJB;
            if (B.n > nmax) nmax = B.n;
            ch.push_back(B);
        }
        if (w > work_cap) { cudaFree(work); work = nullptr; if (cudaMalloc(&work, (size_t)w * sizeof(double)) != cudaSuccess) { rc = PCE_ENOMEM; break; } work_cap = w; }
        if (pz > pan_cap) { cudaFree(panels); panels = nullptr; if (cudaMalloc(&panels, (size_t)pz * sizeof(double)) != cudaSuccess) { rc = PCE_ENOMEM; break; } pan_cap = pz; }
        if ((int)ch.size() > nb_cap) {
            cudaFree(dbod); cudaFree(usum); dbod = nullptr; usum = nullptr;
            if (cudaMalloc(&dbod, ch.size() * sizeof(PcBody)) != cudaSuccess || cudaMalloc(&usum, ch.size() * sizeof(double)) != cudaSuccess) { rc = PCE_ENOMEM; break; }
            nb_cap = (int)ch.size();
        }
        cudaMemcpyAsync(dbod, ch.data(), ch.size() * sizeof(PcBody), cudaMemcpyHostToDevice, c->st);
        const int nch = (int)ch.size();
        // gridDim.z / y are limited to 65535: chunks never hold that many bodies of >= 2 beads within 2^28 elements
        // unless the bodies are tiny; split further if needed
        for (int b0 = 0; b0 < nch; b0 += 32768) {
            const int nbz = (nch - b0 < 32768) ? nch - b0 : 32768;
            const PcBody* bp = dbod + b0;
            k_pc_fill<<<dim3(cdiv(nmax, 16), cdiv(nmax, 16), nbz), 256, 0, c->st>>>(bp, c->rx, c->ry, c->rz, c->p.a, 1.0 / c->p.eps_f, work);
            c->launches++;
            for (int step = 0; step * GJB < nmax; ++step) {
                k_pc_panel<<<dim3(cdiv(nmax, 256), nbz), 256, 0, c->st>>>(bp, step, work, panels);
                k_pc_update<<<dim3(cdiv(nmax, 64), cdiv(nmax, 64), nbz), 256, 0, c->st>>>(bp, step, work, panels);
                c->launches += 2;
            }
            k_pc_rowsum<<<dim3(cdiv(nmax, 8), nbz), 256, 0, c->st>>>(bp, work, u);
            k_pc_usum<<<nbz, 256, 0, c->st>>>(bp, u, usum + b0, c->pc_invs);
            if (c->pc_bf16) k_pc_final<true><<<dim3(cdiv(nmax, 32), cdiv(nmax, 32), nbz), 256, 0, c->st>>>(bp, work, u, usum + b0, c->pc_B);
            else k_pc_final<false><<<dim3(cdiv(nmax, 32), cdiv(nmax, 32), nbz), 256, 0, c->st>>>(bp, work, u, usum + b0, c->pc_B);
            c->launches += 3;
        }
        if (cudaStreamSynchronize(c->st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = PCE_ECUDA; c->err = "preconditioner set-up kernels failed"; }
    }
    cudaFree(work); cudaFree(panels); cudaFree(usum); cudaFree(dbod);
    if (rc == PCE_ENOMEM) {  // not enough room for the work matrices: go without
        cudaGetLastError();
        precond_free(c);
        return PCE_OK;
    }
    if (rc != PCE_OK) return rc;
    c->pc_on = true;
    return PCE_OK;
}

// z_raw = blockdiag(B_i) r  (the caller removes the per-body mean)
int precond_apply(pce_ctx* c, const double* r, double* z)
{
    if (!c->pc_on) return PCE_OK;
    if (c->pc_bf16)
        k_pc_apply<true><<<c->pc_nrows_cta, 256, (size_t)pc_ld(c->pc_max_n) * sizeof(double), c->st>>>((const PcRows*)c->pc_rows, c->pc_B, r, z, c->skip_flag);
    else
        k_pc_apply<false><<<c->pc_nrows_cta, 256, (size_t)pc_ld(c->pc_max_n) * sizeof(double), c->st>>>((const PcRows*)c->pc_rows, c->pc_B, r, z, c->skip_flag);
    c->launches++;
    if (c->pc_nblock < c->Nbody) {
        k_pc_identity<<<cdiv(c->Nbead, 256), 256, 0, c->st>>>(c->Nbead, c->pc_has, c->body_of, 4.0 * PCE_PI * c->p.eps_f * c->p.a, r, z, c->skip_flag);
        c->launches++;
    }
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}
