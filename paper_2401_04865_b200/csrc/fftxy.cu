// fftxy.cu -- the (x, y) transforms of steps 3 and 5 of the spectral Ewald algorithm for cubic-in-(x, y)
// power-of-two meshes, hand-written so that a mesh plane makes ONE trip through HBM per direction.
//
// cuFFT's batched 2-D plans run two kernels per direction (x pass, y pass) and each moves the whole 1 GB array through HBM:
// 4.3 GB per direction at 512^3 for 2.15 GB of algorithmic traffic.  Here one persistent kernel per direction walks the mesh
// plane by plane with two kinds of work items handed out IN ORDER by a global counter:
//   forward:  A(z, a) = real-to-complex x transforms of 2 KP rows of plane z  (reads the real mesh, writes the half spectrum)
//             B(z, b) = complex y transforms of KP columns of plane z, in place in the half spectrum
//   inverse:  B'(z, b) = inverse y transforms, in place;  A'(z, a) = complex-to-real x transforms (writes the real mesh)
// The items of the second kind of plane z are queued DEPTH planes after the first kind and wait on a per-plane arrival counter.
// What the first pass wrote (2.1 MB per plane) is therefore still in the 126 MB L2 when the second pass reads and overwrites it:
// HBM sees one read of the input and one write of the output.  No deadlock: an item only ever waits for items with smaller
// ids, which were claimed earlier by CTAs that never wait.
// x transforms: two real rows a, b as one complex row a + i b (one N-point FFT per row pair), then X_a(k) = (Z(k) + Z*(N-k))/2,
// X_b(k) = (Z(k) - Z*(N-k))/(2i).  FFT: Stockham radix 8 (rest 4 or 2) in shared memory, N/8 threads per transform, KP
// transforms per CTA; the shared tile is [pencil][element] with one pad element per 8 (the first stage writes with stride 8)
// and a pencil stride that puts the pencils of a quarter warp on different banks.
#include "pce_internal.h"
#include "fft_core.h"

#include <cstdlib>

namespace {

using namespace fftcore;

constexpr int DEPTH = 8;   // planes between the two passes of a plane: more items than CTAs in flight, so that waits are rare

template <int N, int NT> struct Geo {
    static constexpr int TP = N / 8;          // threads per transform
    static constexpr int KP = NT / TP;        // transforms per CTA
    static constexpr int PS = N + N / 8 + (KP <= 2 ? 4 : KP <= 4 ? 2 : 1);  // pencil stride (elements)
    static constexpr int NH = N / 2 + 1;
};

__device__ __forceinline__ int pad(int e) { return e + (e >> 3); }

// Pieces of one Stockham stage of radix R on the thread's 8 elements (8 / R butterflies): butterfly q is b = j + q N/8,
// its inputs are the elements b + r N/R, its outputs go to (b - k) R + k + r Ns with k = b mod Ns.
template <int N, int R>
__device__ __forceinline__ int in_index(int j, int q, int r) { return j + q * (N / 8) + r * (N / R); }
template <int N, int R>
__device__ __forceinline__ int out_index(int Ns, int j, int q, int r)
{
    const int b = j + q * (N / 8), k = b & (Ns - 1);
    return (b - k) * R + k + r * Ns;
}
template <int N, int R, int S>
__device__ __forceinline__ void compute_stage(double2* v, int Ns, int j, const double2* __restrict__ tw)
{
#pragma unroll
    for (int q = 0; q < 8 / R; ++q) {
        const int b = j + q * (N / 8);
        twiddle_dft_c<R, S>(v + q * R, tw + tw_offset(Ns), Ns, b & (Ns - 1));
    }
}
template <int N, int R>
__device__ __forceinline__ void load_stage(const double2* pen, int j, double2* v)
{
#pragma unroll
    for (int q = 0; q < 8 / R; ++q)
#pragma unroll
        for (int r = 0; r < R; ++r) v[q * R + r] = pen[pad(in_index<N, R>(j, q, r))];
}
template <int N, int R>
__device__ __forceinline__ void store_stage(double2* pen, int Ns, int j, const double2* v)
{
#pragma unroll
    for (int q = 0; q < 8 / R; ++q)
#pragma unroll
        for (int r = 0; r < R; ++r) pen[pad(out_index<N, R>(Ns, j, q, r))] = v[q * R + r];
}

// barrier over the threads that share a pencil: the whole CTA (WHOLE: a warp touches every pencil) or the N/8 threads of the
// transform (consecutive threads: named barrier 1 + p for two or more warps, else the warp)
template <int N, bool WHOLE>
__device__ __forceinline__ void pencil_sync(int p)
{
    if (WHOLE) __syncthreads();
    else if (N / 8 >= 64) asm volatile("bar.sync %0, %1;" ::"r"(1 + p), "r"(N / 8) : "memory");
    else __syncwarp();
}

// The transform with its first stage fed from registers and its last stage left in registers:
//   in:  v[r] = element j + r N/8 (the inputs of the first radix-8 stage);  out: v[q R + r] = element out_index<N, REST>(N/REST, j, q, r)
// (natural order).  The pencil is scratch; barriers as pencil_sync<N, WHOLE>.
template <int N, int S, bool WHOLE>
__device__ __forceinline__ void fft_regs(double2* v, double2* pen, int p, int j, const double2* __restrict__ tw)
{
    constexpr int REST = Radices<N>::rest, N8 = Radices<N>::n8;
    constexpr int NF8 = (REST == 8) ? N8 - 1 : N8;   // radix-8 stages before the last stage (radix REST)
    compute_stage<N, 8, S>(v, 1, j, tw);
    store_stage<N, 8>(pen, 1, j, v);
    pencil_sync<N, WHOLE>(p);
    int Ns = 8;
#pragma unroll
    for (int st = 1; st < NF8; ++st) {
        load_stage<N, 8>(pen, j, v);
        pencil_sync<N, WHOLE>(p);
        compute_stage<N, 8, S>(v, Ns, j, tw);
        store_stage<N, 8>(pen, Ns, j, v);
        pencil_sync<N, WHOLE>(p);
        Ns *= 8;
    }
    load_stage<N, REST>(pen, j, v);
    compute_stage<N, REST, S>(v, Ns, j, tw);
}

// item id -> (kind, plane, index): slot s holds the n1 first-pass items of plane s (s < nz) and then the n2 second-pass items
// of plane s - DEPTH (s >= DEPTH)
__device__ __forceinline__ void decode_item(int id, int nz, int n1, int n2, int& second, int& z, int& idx)
{
    int s, w;
    const int head = DEPTH * n1;                       // slots 0 .. DEPTH-1: first-pass items only
    const int mid = (nz - DEPTH) * (n1 + n2);          // slots DEPTH .. nz-1: both
    if (id < head) { s = id / n1; w = id % n1; }
    else if (id < head + mid) { const int t = id - head; s = DEPTH + t / (n1 + n2); w = t % (n1 + n2); }
    else { const int t = id - head - mid; s = nz + t / n2; w = n1 + t % n2; }   // slots nz .. nz+DEPTH-1: second-pass items only
    if (s < nz && w < n1) { second = 0; z = s; idx = w; }
    else { second = 1; z = s - DEPTH; idx = w - n1; }
}

__device__ __forceinline__ void wait_plane(const int* done, int want)
{
    if (threadIdx.x == 0) {
        while (*reinterpret_cast<const volatile int*>(done) < want) __nanosleep(100);
        __threadfence();
    }
    __syncthreads();
}

__device__ __forceinline__ void signal_plane(int* done)
{
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) atomicAdd(done, 1);
}

// columns kx0 .. kx0+KP-1 of plane z: N-point transforms along y, in place in the half spectrum.  Thread (j, p), p fastest: a
// warp reads KP consecutive columns (KP x 16 bytes contiguous) of 32 / KP rows; first stage from global memory, last stage to it.
template <int N, int NT, int S>
__device__ __forceinline__ void y_item(double2* gk, int nxh, int z, int b, double2* tile, const double2* __restrict__ tw)
{
    using G = Geo<N, NT>;
    constexpr int REST = Radices<N>::rest;
    const int p = threadIdx.x % G::KP, j = threadIdx.x / G::KP;
    const int kx = b * G::KP + p;
    const bool ok = kx < nxh;
    double2* col = gk + (size_t)z * N * nxh + (ok ? kx : 0);
    double2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) v[r] = __ldcg(col + (size_t)(j + r * G::TP) * nxh);
    fft_regs<N, S, true>(v, tile + p * G::PS, p, j, tw);
    if (ok) {
#pragma unroll
        for (int q = 0; q < 8 / REST; ++q)
#pragma unroll
            for (int r = 0; r < REST; ++r) col[(size_t)out_index<N, REST>(N / REST, j, q, r) * nxh] = v[q * REST + r];
    }
}

// rows 2 KP a .. 2 KP a + 2 KP - 1 of plane z: real -> half-complex along x, two rows per transform.  Thread (p, j), j fastest:
// the N/8 threads of a transform are consecutive, read their two rows coalesced, and synchronise among themselves only.
template <int N, int NT>
__device__ __forceinline__ void x_item_fwd(const double* __restrict__ grid, double2* gk, int nxh, int z, int a, double2* tile,
                                           const double2* __restrict__ tw)
{
    using G = Geo<N, NT>;
    constexpr int REST = Radices<N>::rest;
    const int p = threadIdx.x / G::TP, j = threadIdx.x % G::TP;
    const size_t row = (size_t)z * N + (size_t)a * 2 * G::KP + 2 * p;
    const double* ra = grid + row * N;
    double2* pen = tile + p * G::PS;
    double2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) v[r] = make_double2(__ldg(ra + j + r * G::TP), __ldg(ra + N + j + r * G::TP));
    fft_regs<N, -1, false>(v, pen, p, j, tw);
    pencil_sync<N, false>(p);   // every thread has read its last-stage inputs: the pencil can take the spectrum
#pragma unroll
    for (int q = 0; q < 8 / REST; ++q)
#pragma unroll
        for (int r = 0; r < REST; ++r) pen[pad(out_index<N, REST>(N / REST, j, q, r))] = v[q * REST + r];
    pencil_sync<N, false>(p);
    double2* oa = gk + row * nxh;
    for (int k = j; k <= N / 2; k += G::TP) {
        const double2 Z = pen[pad(k)], Zc = pen[pad((N - k) & (N - 1))];
        oa[k] = make_double2(0.5 * (Z.x + Zc.x), 0.5 * (Z.y - Zc.y));            // X_a = (Z(k) + conj Z(N-k)) / 2
        oa[nxh + k] = make_double2(0.5 * (Z.y + Zc.y), -0.5 * (Z.x - Zc.x));     // X_b = (Z(k) - conj Z(N-k)) / (2i)
    }
}

// the reverse: half-complex rows -> two real rows per transform (unnormalised, as cuFFT's Z2D)
template <int N, int NT>
__device__ __forceinline__ void x_item_inv(const double2* gk, double* __restrict__ grid, int nxh, int z, int a, double2* tile,
                                           const double2* __restrict__ tw)
{
    using G = Geo<N, NT>;
    constexpr int REST = Radices<N>::rest;
    const int p = threadIdx.x / G::TP, j = threadIdx.x % G::TP;
    const size_t row = (size_t)z * N + (size_t)a * 2 * G::KP + 2 * p;
    const double2* ia = gk + row * nxh;
    double2* pen = tile + p * G::PS;
    for (int k = j; k <= N / 2; k += G::TP) {
        double2 A = __ldcg(ia + k), B = __ldcg(ia + nxh + k);
        if (k == 0 || k == N / 2) { A.y = 0.0; B.y = 0.0; }  // the imaginary parts of the self-conjugate modes carry no information
        pen[pad(k)] = make_double2(A.x - B.y, A.y + B.x);                              // Z(k) = X_a + i X_b
        if (k > 0 && k < N / 2) pen[pad(N - k)] = make_double2(A.x + B.y, B.x - A.y);  // Z(N-k) = conj X_a + i conj X_b
    }
    pencil_sync<N, false>(p);
    double2 v[8];
    load_stage<N, 8>(pen, j, v);
    pencil_sync<N, false>(p);
    fft_regs<N, +1, false>(v, pen, p, j, tw);
    double* ra = grid + row * N;
#pragma unroll
    for (int q = 0; q < 8 / REST; ++q)
#pragma unroll
        for (int r = 0; r < REST; ++r) {
            const int e = out_index<N, REST>(N / REST, j, q, r);
            ra[e] = v[q * REST + r].x;
            ra[N + e] = v[q * REST + r].y;
        }
}

// ctr[0]: work counter; ctr[1 + z]: arrivals of the first pass of plane z (both zeroed before the launch)
template <int N, int NT, bool INVERSE>
__global__ void __launch_bounds__(NT, 1024 / NT)
k_fft_xy(const double* gin, double* gout, double2* gk, int nz, const double2* __restrict__ tw_g, int* __restrict__ ctr,
         const int* __restrict__ skip)
{
    if (skip && *skip) return;
    using G = Geo<N, NT>;
    extern __shared__ __align__(16) unsigned char fsm[];
    double2* tile = reinterpret_cast<double2*>(fsm);   // [KP][PS]
    double2* tw = tile + G::KP * G::PS;                // per-stage twiddle tables
    __shared__ int s_item;
    for (int i = threadIdx.x; i < TwSize<N>::value; i += NT) tw[i] = tw_g[i];
    constexpr int nxh = G::NH;
    constexpr int nX = N / (2 * G::KP), nY = (nxh + G::KP - 1) / G::KP;
    constexpr int n1 = INVERSE ? nY : nX, n2 = INVERSE ? nX : nY;
    const int total = nz * (n1 + n2);
    // inverse: the rows an x item has consumed are dead (as with cuFFT's Z2D the spectrum does not survive); telling L2 so saves
    // their write-back -- the y pass left them dirty in L2 and they never need to reach HBM
    constexpr size_t blk_bytes = (size_t)2 * G::KP * nxh * sizeof(double2);
    constexpr bool can_discard = INVERSE && (blk_bytes % 128 == 0);
    unsigned char* dead = nullptr;
    for (;;) {
        __syncthreads();
        if (can_discard && dead) {
            for (size_t o = (size_t)threadIdx.x * 128; o < blk_bytes; o += (size_t)NT * 128)
                asm volatile("discard.global.L2 [%0], 128;" ::"l"(dead + o) : "memory");
            dead = nullptr;
        }
        if (threadIdx.x == 0) s_item = atomicAdd(&ctr[0], 1);
        __syncthreads();
        const int id = s_item;
        if (id >= total) break;
        int second, z, idx;
        decode_item(id, nz, n1, n2, second, z, idx);
        if (!second) {
            if (INVERSE) y_item<N, NT, +1>(gk, nxh, z, idx, tile, tw);
            else x_item_fwd<N, NT>(gin, gk, nxh, z, idx, tile, tw);
            signal_plane(&ctr[1 + z]);
        } else {
            wait_plane(&ctr[1 + z], n1);
            if (INVERSE) {
                x_item_inv<N, NT>(gk, gout, nxh, z, idx, tile, tw);
                dead = reinterpret_cast<unsigned char*>(gk + ((size_t)z * N + (size_t)idx * 2 * G::KP) * nxh);
            }
            else y_item<N, NT, -1>(gk, nxh, z, idx, tile, tw);
        }
    }
}

template <int N, int NT> size_t smem_of() { return (size_t)(Geo<N, NT>::KP * Geo<N, NT>::PS + TwSize<N>::value) * sizeof(double2); }

template <int N, int NT, bool INVERSE> int launch_one(pce_ctx* c, cufftDoubleComplex* gk)
{
    using G = Geo<N, NT>;
    const size_t smem = smem_of<N, NT>();
    const int nz = c->wk.Ng[2];
    int& occ = c->xy_occ[INVERSE ? 1 : 0];
    if (occ == 0) {  // first use on this context: raise the shared-memory limit, size the persistent grid
        PCE_CUDA(c, cudaFuncSetAttribute(k_fft_xy<N, NT, INVERSE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_fft_xy<N, NT, INVERSE>, NT, smem));
        if (occ < 1) { c->err = "fftxy kernels do not fit on this device"; return PCE_ECUDA; }
    }
    PCE_CUDA(c, cudaMemsetAsync(c->xy_ctr, 0, ((size_t)nz + 1) * sizeof(int), c->st));
    const int total = nz * (N / (2 * G::KP) + (G::NH + G::KP - 1) / G::KP);
    int blocks = c->num_sm * occ;
    if (blocks > total) blocks = total;
    k_fft_xy<N, NT, INVERSE><<<blocks, NT, smem, c->st>>>(INVERSE ? nullptr : c->grid, INVERSE ? c->grid : nullptr, reinterpret_cast<double2*>(gk),
                                                         nz, c->xytw, c->xy_ctr, c->skip_flag);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

template <int N, bool INVERSE> int launch_xy(pce_ctx* c, cufftDoubleComplex* gk)
{
    if (c->xy_nt[INVERSE ? 1 : 0] == 128) return launch_one<N, 128, INVERSE>(c, gk);
    if (c->xy_nt[INVERSE ? 1 : 0] == 512) return launch_one<N, 512, INVERSE>(c, gk);
    return launch_one<N, 256, INVERSE>(c, gk);
}

}  // namespace

// own (x, y) transforms: N_x = N_y a power of two in 128..1024, at least DEPTH planes, fused z pass in use
bool fftxy_supported(const pce_params& p)
{
    const int n = p.Ng[0];
    if (p.Ng[1] != n || !(n == 128 || n == 256 || n == 512 || n == 1024) || p.Ng[2] < DEPTH) return false;
    const char* e = getenv("PCE_NO_FFTXY");
    return !(e && e[0] == '1');
}

int fftxy_init(pce_ctx* c)
{
    const int n = c->p.Ng[0];
    std::vector<double2> tw;
    stage_twiddles(n, tw);
    PCE_CUDA(c, cudaMalloc(&c->xytw, tw.size() * sizeof(double2)));
    PCE_CUDA(c, cudaMemcpy(c->xytw, tw.data(), tw.size() * sizeof(double2), cudaMemcpyHostToDevice));
    PCE_CUDA(c, cudaMalloc(&c->xy_ctr, ((size_t)c->p.Ng[2] + 1) * sizeof(int)));
    // threads per CTA of the forward / inverse kernel: 256 (measured best at 512^3: 0.79 / 0.89 ms; 128 threads 1.00 / 1.15 ms,
    // 512 threads 0.83 / 0.93 ms); the environment variables select the other instantiations for tuning on other meshes
    const char* ef = getenv("PCE_FFTXY_NT_F");
    const char* ei = getenv("PCE_FFTXY_NT_I");
    c->xy_nt[0] = (ef && (atoi(ef) == 128 || atoi(ef) == 512)) ? atoi(ef) : 256;
    c->xy_nt[1] = (ei && (atoi(ei) == 128 || atoi(ei) == 512)) ? atoi(ei) : 256;
    c->xy_occ[0] = c->xy_occ[1] = 0;
    return PCE_OK;
}

int fftxy_forward(pce_ctx* c, cufftDoubleComplex* gk)
{
    switch (c->p.Ng[0]) {
        case 128: return launch_xy<128, false>(c, gk);
        case 256: return launch_xy<256, false>(c, gk);
        case 512: return launch_xy<512, false>(c, gk);
        default: return launch_xy<1024, false>(c, gk);
    }
}

int fftxy_inverse(pce_ctx* c, cufftDoubleComplex* gk)
{
    switch (c->p.Ng[0]) {
        case 128: return launch_xy<128, true>(c, gk);
        case 256: return launch_xy<256, true>(c, gk);
        case 512: return launch_xy<512, true>(c, gk);
        default: return launch_xy<1024, true>(c, gk);
    }
}
