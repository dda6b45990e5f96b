// fft_kernels.cu -- the four FFT kernels of the hot path (stages S1, S2, S4, S5 of DESIGN.md)
// and their full-input fp64 variants used once by hfft_build_tensor for the tensor bank.
//
//   S1 fftx_fwd : M = Ms_j m (Eq.17), real-to-complex DFT of length 2nx of a row that
//                 is zero beyond nx (F_1 of Eq.23), kept for kx = 0..nx, stored
//                 TRANSPOSED so that the y transforms work on contiguous rows
//   S2 ffty_fwd : complex DFT of length 2ny along y (F_2 of Eq.24), rows >= ny zero
//   S4 iffty    : inverse along y, only the first ny outputs (crop fused)
//   S5 ifftx    : complex-to-real inverse of length 2nx, only the first nx outputs
//
// Layouts (C = complex of T):
//   real field      [plane][rows][nx]           plane = (state, component, layer)
//   X^ (after S1)   [plane][nx+1][rows] C       (kx major, y fastest)
//   M^ (after S2)   [plane][KS] C, element k = kx * 2ny + ky
// The z-component planes of M^ hold i*M_z (and H^ holds i*H_z) so that the layer coupling is a
// real matrix acting on real and imaginary parts alike.
#include "hfft_internal.h"
#include "fft.cuh"

namespace hfft {

// ------------------------------------------------------------------------------------------
// S1: forward x.  A real row of 2N samples (only the first N non-zero if ZP) is packed as N
// complex z[t] = x[2t] + i x[2t+1]; Z = DFT_N(z); X[k] = E[k] + W_2N^k O[k] with
// E = (Z[k] + conj Z[N-k]) / 2, O = (Z[k] - conj Z[N-k]) / (2i).
// One CTA = RB consecutive rows (y) of one plane; the split post-processing runs with lanes
// along y so that every store to the transposed X^ is a run of RB consecutive elements.
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2N, bool ZP>
__global__ void __launch_bounds__(1024)
fftx_fwd_kernel(const T* __restrict__ in, HFFT_C* __restrict__ xhat, int rb, int rows_per_plane, int nz, int use_ms,
                MsParam<T> ms, const HFFT_C* __restrict__ tw /* exp(-2 pi i t / 2N), 2N entries */) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, false, ZP> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR, PITCH = N + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);
    const long long row0 = (long long)blockIdx.x * rb;          // global row index (plane * rows + y)
    const int plane = (int)(row0 / rows_per_plane);
    const int y0 = (int)(row0 - (long long)plane * rows_per_plane);
    const C* zin = reinterpret_cast<const C*>(in) + (row0 + r) * (ZP ? N / 2 : N);
    C v[R];
    constexpr int RL = (ZP && R > 1) ? R / 2 : R;
#pragma unroll
    for (int q = 0; q < RL; ++q) v[q] = zin[j + q * TPR];
    if (ZP && use_ms) {
        const T sc = ms.v[plane % nz];
#pragma unroll
        for (int q = 0; q < RL; ++q) { v[q].x *= sc; v[q].y *= sc; }
    }
    C* srow = s + r * PITCH;
    F::run(v, srow, j, tw, 2);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < R; ++q) srow[swz(j + q * TPR)] = v[q];
    __syncthreads();

    // post-process: pairs (k, N-k), k = 0..N/2, lanes along the rb rows
    C* xp = xhat + (long long)plane * (N + 1) * rows_per_plane + y0;
    const int nthreads = blockDim.x;
    for (int w = tid; w < (N / 2 + 1) * rb; w += nthreads) {
        const int k = w / rb, rr = w - k * rb;
        const C* sr = s + rr * PITCH;
        if (k == 0) {
            C z0 = sr[0];
            xp[rr] = mk<T>(z0.x + z0.y, 0);
            xp[(long long)N * rows_per_plane + rr] = mk<T>(z0.x - z0.y, 0);
        } else {
            C zk = sr[swz(k)], zn = sr[swz(N - k)];
            C E = mk<T>((zk.x + zn.x) * (T)0.5, (zk.y - zn.y) * (T)0.5);
            C O = mk<T>((zk.y + zn.y) * (T)0.5, (zn.x - zk.x) * (T)0.5);
            C WO = cmul(__ldg(tw + k), O);
            xp[(long long)k * rows_per_plane + rr] = cadd(E, WO);
            if (k != N - k) xp[(long long)(N - k) * rows_per_plane + rr] = cconj(csub(E, WO));
        }
    }
}

// ------------------------------------------------------------------------------------------
// S5: inverse x (complex-to-real, crop to the first N reals = first N/2 complex outputs).
// Z~[k] = E~ + i O~,  E~ = X[k] + conj X[N-k],  O~ = (X[k] - conj X[N-k]) W_2N^{-k};
// z~ = IDFT_N(Z~) holds x~[2t] + i x~[2t+1].  Same CTA shape as S1: the pre-processing reads the
// transposed X^ with lanes along y.
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2N>
__global__ void __launch_bounds__(1024)
ifftx_kernel(const HFFT_C* __restrict__ xhat, T* __restrict__ out, int rb, int rows_per_plane,
             const HFFT_C* __restrict__ tw) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, true, false> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR, PITCH = N + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);
    const long long row0 = (long long)blockIdx.x * rb;
    const int plane = (int)(row0 / rows_per_plane);
    const int y0 = (int)(row0 - (long long)plane * rows_per_plane);
    const C* xp = xhat + (long long)plane * (N + 1) * rows_per_plane + y0;
    const int nthreads = blockDim.x;
    for (int w = tid; w < (N / 2 + 1) * rb; w += nthreads) {
        const int k = w / rb, rr = w - k * rb;
        C* sr = s + rr * PITCH;
        C xk = xp[(long long)k * rows_per_plane + rr];
        C xn = xp[(long long)(N - k) * rows_per_plane + rr];      // k = 0: the Nyquist row kx = N
        C E = mk<T>(xk.x + xn.x, xk.y - xn.y);
        C D = mk<T>(xk.x - xn.x, xk.y + xn.y);
        C O = (k == 0) ? D : cmulc(D, __ldg(tw + k));
        // Z~[k] = E + i O ; Z~[N-k] = conj(E) + i conj(O)
        sr[swz(k)] = mk<T>(E.x - O.y, E.y + O.x);
        if (k != 0 && k != N - k) sr[swz(N - k)] = mk<T>(E.x + O.y, O.x - E.y);
    }
    __syncthreads();
    C* srow = s + r * PITCH;
    C v[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = srow[swz(j + q * TPR)];
    F::run(v, srow, j, tw, 2);
    C* zout = reinterpret_cast<C*>(out) + (row0 + r) * (N / 2);
    constexpr int RS = R > 1 ? R / 2 : 1;
#pragma unroll
    for (int q = 0; q < RS; ++q) zout[j + q * TPR] = v[q];
}

// ------------------------------------------------------------------------------------------
// S2 / S4: transforms along y on the contiguous rows of the transposed X^.  Row = (plane, kx);
// a CTA handles `rpc` consecutive rows, TPR threads per row.
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2N, bool ZP>
__global__ void __launch_bounds__(256)
ffty_fwd_kernel(const HFFT_C* __restrict__ xhat, HFFT_C* __restrict__ spec, long long nrows, int nxp1, int nz_rot,
                long long ks, const HFFT_C* __restrict__ tw /* N entries */) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, false, ZP> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);
    const int rpc = blockDim.x >> F::LOG2TPR;
    const long long row = (long long)blockIdx.x * rpc + r;
    const bool live = row < nrows;
    const long long rowc = live ? row : nrows - 1;
    const C* zin = xhat + rowc * (ZP ? N / 2 : N);
    C v[R];
    constexpr int RL = ZP ? R / 2 : R;
#pragma unroll
    for (int q = 0; q < RL; ++q) v[q] = zin[j + q * TPR];
    F::run(v, s + r * N, j, tw, 1);
    if (!live) return;
    const int plane = (int)(row / nxp1);
    const int kx = (int)(row - (long long)plane * nxp1);
    if (nz_rot > 0 && (plane / nz_rot) % 3 == 2) {   // M'_z = i M_z
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = mul_pi(v[q]);
    }
    C* dst = spec + (long long)plane * ks + (long long)kx * N;
#pragma unroll
    for (int q = 0; q < R; ++q) dst[j + q * TPR] = v[q];
}

template <typename T, int LOG2N>
__global__ void __launch_bounds__(256)
iffty_kernel(const HFFT_C* __restrict__ spec, HFFT_C* __restrict__ xhat, long long nrows, int nxp1, int nz_rot,
             long long ks, const HFFT_C* __restrict__ tw) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, true, false> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);
    const int rpc = blockDim.x >> F::LOG2TPR;
    const long long row = (long long)blockIdx.x * rpc + r;
    const bool live = row < nrows;
    const long long rowc = live ? row : nrows - 1;
    const int plane = (int)(rowc / nxp1);
    const int kx = (int)(rowc - (long long)plane * nxp1);
    const C* src = spec + (long long)plane * ks + (long long)kx * N;
    C v[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = src[j + q * TPR];
    if (nz_rot > 0 && (plane / nz_rot) % 3 == 2) {   // H_z = -i H'_z
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = mul_mi(v[q]);
    }
    F::run(v, s + r * N, j, tw, 1);
    if (!live) return;
    C* dst = xhat + row * (N / 2);
#pragma unroll
    for (int q = 0; q < R / 2; ++q) dst[j + q * TPR] = v[q];
}

// ------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------
// opt in to > 48 KB of dynamic shared memory once per kernel instantiation (`done` is a static
// local of the dispatch case, i.e. one flag per instantiation)
template <typename K> static cudaError_t set_smem(K kernel, size_t bytes, size_t& done) {
    if (bytes <= 48 * 1024 || bytes <= done) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) done = bytes;
    return e;
}

#define HFFT_CASE(V, ...) case V: { constexpr int L = V; __VA_ARGS__ } break;
#define HFFT_DISPATCH_X(LG, ...)                                                                    \
    switch (LG) {                                                                                   \
        HFFT_CASE(1, __VA_ARGS__) HFFT_CASE(2, __VA_ARGS__) HFFT_CASE(3, __VA_ARGS__) HFFT_CASE(4, __VA_ARGS__) \
        HFFT_CASE(5, __VA_ARGS__) HFFT_CASE(6, __VA_ARGS__) HFFT_CASE(7, __VA_ARGS__) HFFT_CASE(8, __VA_ARGS__) \
        HFFT_CASE(9, __VA_ARGS__) HFFT_CASE(10, __VA_ARGS__)                                        \
        default: break;                                                                             \
    }
#define HFFT_DISPATCH_Y(LG, ...)                                                                    \
    switch (LG) {                                                                                   \
        HFFT_CASE(2, __VA_ARGS__) HFFT_CASE(3, __VA_ARGS__) HFFT_CASE(4, __VA_ARGS__) HFFT_CASE(5, __VA_ARGS__) \
        HFFT_CASE(6, __VA_ARGS__) HFFT_CASE(7, __VA_ARGS__) HFFT_CASE(8, __VA_ARGS__) HFFT_CASE(9, __VA_ARGS__) \
        HFFT_CASE(10, __VA_ARGS__) HFFT_CASE(11, __VA_ARGS__)                                       \
        default: break;                                                                             \
    }

// rows per CTA of the x kernels: a 128-byte run of the transposed X^, at most 1024 threads
template <typename T> static int x_rows_per_cta(int log2N, int rows_per_plane) {
    const int tpr = (1 << log2N) / (log2N < 3 ? (1 << log2N) : 8);
    int rb = (int)(128 / sizeof(HFFT_C));
    while (rb > 1 && rb * tpr > 1024) rb /= 2;
    if (rb > rows_per_plane) rb = rows_per_plane;
    return rb;
}

template <typename T, bool ZP>
cudaError_t launch_fftx_fwd(const T* in, void* xhat, int log2nx, int nplanes, int rows_per_plane, int nz,
                            const double* ms_host, const void* tw, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2nx;
    const int rb = x_rows_per_cta<T>(log2nx, rows_per_plane);
    const int tpr = N / (log2nx < 3 ? N : 8);
    const size_t smem = (size_t)rb * (N + 1) * sizeof(C);
    const long long grid = (long long)nplanes * rows_per_plane / rb;
    MsParam<T> ms;
    const int use_ms = ms_host != nullptr;
    for (int k = 0; k < HFFT_MAX_NZ; ++k) ms.v[k] = (use_ms && k < nz) ? (T)ms_host[k] : (T)1;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_X(log2nx, {
        auto kern = fftx_fwd_kernel<T, L, ZP>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<(unsigned)grid, rb * tpr, smem, st>>>(in, (C*)xhat, rb, rows_per_plane, nz > 0 ? nz : 1, use_ms, ms,
                                                         (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_ifftx(const void* xhat, T* out, int log2nx, int nplanes, int rows_per_plane, const void* tw,
                         cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2nx;
    const int rb = x_rows_per_cta<T>(log2nx, rows_per_plane);
    const int tpr = N / (log2nx < 3 ? N : 8);
    const size_t smem = (size_t)rb * (N + 1) * sizeof(C);
    const long long grid = (long long)nplanes * rows_per_plane / rb;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_X(log2nx, {
        auto kern = ifftx_kernel<T, L>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<(unsigned)grid, rb * tpr, smem, st>>>((const C*)xhat, out, rb, rows_per_plane, (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

template <typename T, bool ZP>
cudaError_t launch_ffty_fwd(const void* xhat, void* spec, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                            const void* tw, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2N;
    const int tpr = log2N < 3 ? 1 : N / 8;
    const int rpc = tpr >= 256 ? 1 : 256 / tpr;
    const long long nrows = (long long)nplanes * (nx + 1);
    const size_t smem = (size_t)rpc * N * sizeof(C);
    const long long grid = (nrows + rpc - 1) / rpc;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_Y(log2N, {
        auto kern = ffty_fwd_kernel<T, L, ZP>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<(unsigned)grid, rpc * tpr, smem, st>>>((const C*)xhat, (C*)spec, nrows, nx + 1, nz_rot, ks,
                                                          (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_iffty(const void* spec, void* xhat, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                         const void* tw, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2N;
    const int tpr = log2N < 3 ? 1 : N / 8;
    const int rpc = tpr >= 256 ? 1 : 256 / tpr;
    const long long nrows = (long long)nplanes * (nx + 1);
    const size_t smem = (size_t)rpc * N * sizeof(C);
    const long long grid = (nrows + rpc - 1) / rpc;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_Y(log2N, {
        auto kern = iffty_kernel<T, L>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<(unsigned)grid, rpc * tpr, smem, st>>>((const C*)spec, (C*)xhat, nrows, nx + 1, nz_rot, ks,
                                                          (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

// explicit instantiations used by hfft_api.cu / tensor_build.cu
template cudaError_t launch_fftx_fwd<float, true>(const float*, void*, int, int, int, int, const double*, const void*, cudaStream_t);
template cudaError_t launch_fftx_fwd<double, true>(const double*, void*, int, int, int, int, const double*, const void*, cudaStream_t);
template cudaError_t launch_fftx_fwd<double, false>(const double*, void*, int, int, int, int, const double*, const void*, cudaStream_t);
template cudaError_t launch_ifftx<float>(const void*, float*, int, int, int, const void*, cudaStream_t);
template cudaError_t launch_ifftx<double>(const void*, double*, int, int, int, const void*, cudaStream_t);
template cudaError_t launch_ffty_fwd<float, true>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_ffty_fwd<double, true>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_ffty_fwd<double, false>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_iffty<float>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_iffty<double>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);

}  // namespace hfft
