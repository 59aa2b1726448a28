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

namespace {

using namespace fftcore;

constexpr int NT = 256;    // threads per CTA
constexpr int DEPTH = 2;   // planes between the two passes of a plane

template <int N> struct Geo {
    static constexpr int TP = N / 8;          // threads per transform
    static constexpr int KP = NT / TP;        // transforms per CTA
    static constexpr int PS = N + N / 8 + (KP <= 2 ? 4 : KP <= 4 ? 2 : 1);  // pencil stride (elements)
    static constexpr int NH = N / 2 + 1;
};

__device__ __forceinline__ int pad(int e) { return e + (e >> 3); }

// one Stockham stage of radix R on the thread's 8 elements, in place in the padded pencil (barrier between loads and stores)
template <int N, int R, int S>
__device__ __forceinline__ void sstage(double2* pen, int Ns, int j, const double2* __restrict__ tw)
{
    constexpr int NB = 8 / R, TP = N / 8;
    double2 v[8];
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = j + q * TP;
#pragma unroll
        for (int r = 0; r < R; ++r) v[q * R + r] = pen[pad(b + r * (N / R))];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int b = j + q * TP;
        const int k = b & (Ns - 1);
        twiddle_dft<R, S>(v + q * R, k * (N / (Ns * R)), tw);
        const int d = (b - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) pen[pad(d + r * Ns)] = v[q * R + r];
    }
    __syncthreads();
}

// N-point transform of the pencil (natural order in and out); the data must be in place and visible (barrier before the call)
template <int N, int S>
__device__ __forceinline__ void fft_smem(double2* pen, int j, const double2* __restrict__ tw)
{
    constexpr int REST = Radices<N>::rest, N8 = Radices<N>::n8;
    constexpr int NF8 = (REST == 8) ? N8 - 1 : N8;
    int Ns = 1;
    if (NF8 >= 1) { sstage<N, 8, S>(pen, Ns, j, tw); Ns *= 8; }
    if (NF8 >= 2) { sstage<N, 8, S>(pen, Ns, j, tw); Ns *= 8; }
    if (NF8 >= 3) { sstage<N, 8, S>(pen, Ns, j, tw); Ns *= 8; }
    sstage<N, REST, S>(pen, Ns, j, tw);
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

// columns kx0 .. kx0+KP-1 of plane z: N-point transforms along y, in place in the half spectrum
template <int N, int S>
__device__ __forceinline__ void y_item(double2* gk, int nxh, int z, int b, double2* tile, const double2* __restrict__ tw)
{
    using G = Geo<N>;
    const int p = threadIdx.x % G::KP, j = threadIdx.x / G::KP;
    const int kx = b * G::KP + p;
    const bool ok = kx < nxh;
    double2* col = gk + (size_t)z * N * nxh + (ok ? kx : 0);
    double2* pen = tile + p * G::PS;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int y = j + r * G::TP;
        pen[pad(y)] = ok ? __ldcg(col + (size_t)y * nxh) : make_double2(0.0, 0.0);
    }
    __syncthreads();
    fft_smem<N, S>(pen, j, tw);
    if (ok) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int y = j + r * G::TP;
            col[(size_t)y * nxh] = pen[pad(y)];
        }
    }
    __syncthreads();
}

// rows 2 KP a .. 2 KP a + 2 KP - 1 of plane z: real -> half-complex along x (two rows per transform)
template <int N>
__device__ __forceinline__ void x_item_fwd(const double* __restrict__ grid, double2* gk, int nxh, int z, int a, double2* tile,
                                           const double2* __restrict__ tw)
{
    using G = Geo<N>;
    const size_t row0 = (size_t)z * N + (size_t)a * 2 * G::KP;
    for (int i = threadIdx.x; i < G::KP * N; i += NT) {  // consecutive lanes: consecutive x of one row pair
        const int pp = i / N, e = i % N;
        const double* ra = grid + (row0 + 2 * pp) * N;
        tile[pp * G::PS + pad(e)] = make_double2(__ldg(ra + e), __ldg(ra + N + e));
    }
    __syncthreads();
    fft_smem<N, -1>(tile + (threadIdx.x % G::KP) * G::PS, threadIdx.x / G::KP, tw);
    for (int i = threadIdx.x; i < G::KP * G::NH; i += NT) {
        const int pp = i / G::NH, k = i % G::NH;
        const double2 Z = tile[pp * G::PS + pad(k)], Zc = tile[pp * G::PS + pad((N - k) & (N - 1))];
        double2* oa = gk + (row0 + 2 * pp) * nxh + k;
        oa[0] = make_double2(0.5 * (Z.x + Zc.x), 0.5 * (Z.y - Zc.y));      // X_a = (Z(k) + conj Z(N-k)) / 2
        oa[nxh] = make_double2(0.5 * (Z.y + Zc.y), -0.5 * (Z.x - Zc.x));   // X_b = (Z(k) - conj Z(N-k)) / (2i)
    }
    __syncthreads();
}

// the reverse: half-complex rows -> two real rows per transform (unnormalised, as cuFFT's Z2D)
template <int N>
__device__ __forceinline__ void x_item_inv(const double2* gk, double* __restrict__ grid, int nxh, int z, int a, double2* tile,
                                           const double2* __restrict__ tw)
{
    using G = Geo<N>;
    const size_t row0 = (size_t)z * N + (size_t)a * 2 * G::KP;
    for (int i = threadIdx.x; i < G::KP * G::NH; i += NT) {
        const int pp = i / G::NH, k = i % G::NH;
        const double2* ia = gk + (row0 + 2 * pp) * nxh + k;
        double2 A = __ldcg(ia), B = __ldcg(ia + nxh);
        if (k == 0 || k == N / 2) { A.y = 0.0; B.y = 0.0; }  // the imaginary parts of the self-conjugate modes carry no information
        double2* pen = tile + pp * G::PS;
        pen[pad(k)] = make_double2(A.x - B.y, A.y + B.x);                          // Z(k) = X_a + i X_b
        if (k > 0 && k < N / 2) pen[pad(N - k)] = make_double2(A.x + B.y, B.x - A.y);  // Z(N-k) = conj X_a + i conj X_b
    }
    __syncthreads();
    fft_smem<N, +1>(tile + (threadIdx.x % G::KP) * G::PS, threadIdx.x / G::KP, tw);
    for (int i = threadIdx.x; i < G::KP * N; i += NT) {
        const int pp = i / N, e = i % N;
        const double2 v = tile[pp * G::PS + pad(e)];
        double* ra = grid + (row0 + 2 * pp) * N;
        ra[e] = v.x;
        ra[N + e] = v.y;
    }
    __syncthreads();
}

// ctr[0]: work counter; ctr[1 + z]: arrivals of the first pass of plane z (both zeroed before the launch)
template <int N, bool INVERSE>
__global__ void __launch_bounds__(NT, 3)
k_fft_xy(const double* gin, double* gout, double2* gk, int nz, const double2* __restrict__ tw_g, int* __restrict__ ctr,
         const int* __restrict__ skip)
{
    if (skip && *skip) return;
    using G = Geo<N>;
    extern __shared__ __align__(16) unsigned char fsm[];
    double2* tile = reinterpret_cast<double2*>(fsm);   // [KP][PS]
    double2* tw = tile + G::KP * G::PS;                // [N]
    __shared__ int s_item;
    for (int i = threadIdx.x; i < N; i += NT) tw[i] = tw_g[i];
    constexpr int nxh = G::NH;
    constexpr int nX = N / (2 * G::KP), nY = (nxh + G::KP - 1) / G::KP;
    constexpr int n1 = INVERSE ? nY : nX, n2 = INVERSE ? nX : nY;
    const int total = nz * (n1 + n2);
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(&ctr[0], 1);
        __syncthreads();
        const int id = s_item;
        if (id >= total) break;
        int second, z, idx;
        decode_item(id, nz, n1, n2, second, z, idx);
        if (!second) {
            if (INVERSE) y_item<N, +1>(gk, nxh, z, idx, tile, tw);
            else x_item_fwd<N>(gin, gk, nxh, z, idx, tile, tw);
            signal_plane(&ctr[1 + z]);
        } else {
            wait_plane(&ctr[1 + z], n1);
            if (INVERSE) x_item_inv<N>(gk, gout, nxh, z, idx, tile, tw);
            else y_item<N, -1>(gk, nxh, z, idx, tile, tw);
        }
    }
}

template <int N> size_t smem_of() { return (size_t)(Geo<N>::KP * Geo<N>::PS + N) * sizeof(double2); }

template <int N> int launch_xy(pce_ctx* c, bool inverse, cufftDoubleComplex* gk)
{
    const size_t smem = smem_of<N>();
    const int nz = c->wk.Ng[2];
    PCE_CUDA(c, cudaMemsetAsync(c->xy_ctr, 0, ((size_t)nz + 1) * sizeof(int), c->st));
    const int total = nz * (N / (2 * Geo<N>::KP) + (Geo<N>::NH + Geo<N>::KP - 1) / Geo<N>::KP);
    int blocks = c->num_sm * c->xy_occ;
    if (blocks > total) blocks = total;
    if (inverse)
        k_fft_xy<N, true><<<blocks, NT, smem, c->st>>>(nullptr, c->grid, reinterpret_cast<double2*>(gk), nz, c->xytw, c->xy_ctr, c->skip_flag);
    else
        k_fft_xy<N, false><<<blocks, NT, smem, c->st>>>(c->grid, nullptr, reinterpret_cast<double2*>(gk), nz, c->xytw, c->xy_ctr, c->skip_flag);
    c->launches++;
    PCE_CUDA(c, cudaGetLastError());
    return PCE_OK;
}

template <int N> int init_xy(pce_ctx* c)
{
    const int smem = (int)smem_of<N>();
    PCE_CUDA(c, cudaFuncSetAttribute(k_fft_xy<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    PCE_CUDA(c, cudaFuncSetAttribute(k_fft_xy<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int o1 = 0, o2 = 0;
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o1, k_fft_xy<N, true>, NT, smem));
    PCE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o2, k_fft_xy<N, false>, NT, smem));
    c->xy_occ = o1 < o2 ? o1 : o2;
    if (c->xy_occ < 1) { c->err = "fftxy kernels do not fit on this device"; return PCE_ECUDA; }
    return PCE_OK;
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
    std::vector<double2> tw(n);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int m = 0; m < n; ++m) tw[m] = make_double2((double)cosl(-2.0L * pi * m / n), (double)sinl(-2.0L * pi * m / n));
    PCE_CUDA(c, cudaMalloc(&c->xytw, n * sizeof(double2)));
    PCE_CUDA(c, cudaMemcpy(c->xytw, tw.data(), n * sizeof(double2), cudaMemcpyHostToDevice));
    PCE_CUDA(c, cudaMalloc(&c->xy_ctr, ((size_t)c->p.Ng[2] + 1) * sizeof(int)));
    switch (n) {
        case 128: return init_xy<128>(c);
        case 256: return init_xy<256>(c);
        case 512: return init_xy<512>(c);
        default: return init_xy<1024>(c);
    }
}

int fftxy_forward(pce_ctx* c, cufftDoubleComplex* gk)
{
    switch (c->p.Ng[0]) {
        case 128: return launch_xy<128>(c, false, gk);
        case 256: return launch_xy<256>(c, false, gk);
        case 512: return launch_xy<512>(c, false, gk);
        default: return launch_xy<1024>(c, false, gk);
    }
}

int fftxy_inverse(pce_ctx* c, cufftDoubleComplex* gk)
{
    switch (c->p.Ng[0]) {
        case 128: return launch_xy<128>(c, true, gk);
        case 256: return launch_xy<256>(c, true, gk);
        case 512: return launch_xy<512>(c, true, gk);
        default: return launch_xy<1024>(c, true, gk);
    }
}
