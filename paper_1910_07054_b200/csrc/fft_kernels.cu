// fft_kernels.cu -- the four FFT kernels of the hot path (stages S1, S2, S4, S5 of DESIGN.md)
// and their full-input fp64 variants used once by hfft_build_tensor for the tensor bank.
//
//   S1 fftx_fwd : M = Ms_j m (Eq.17), real-to-complex DFT of length 2nx of a row that
//                 is zero beyond nx (F_1 of Eq.23), kept for kx = 0..nx
//   S2 ffty_fwd : complex DFT of length 2ny along y (F_2 of Eq.24), rows >= ny zero
//   S4 iffty    : inverse along y, only the first ny outputs (crop fused)
//   S5 ifftx    : complex-to-real inverse of length 2nx, only the first nx outputs
//
// Layouts (C = complex of T):
//   real field      [plane][rows][nx]           plane = (state, component, layer)
//   X^ (after S1)   main [plane*rows][nx] C, then Nyquist column kx = nx: [plane*rows] C
//   M^ (after S2)   [plane][KS] C, element k = ky*nx + kx (kx < nx), 2ny*nx + ky (kx = nx)
// The z-component planes of M^ hold i*M_z (and H^ holds i*H_z) so that the layer coupling is a
// real matrix acting on real and imaginary parts alike.
#include "hfft_internal.h"
#include "fft.cuh"

namespace hfft {

static constexpr int kThreads = 256;

// ------------------------------------------------------------------------------------------
// S1: forward x.  A real row of 2N samples (only the first N non-zero if ZP) is packed as N
// complex z[t] = x[2t] + i x[2t+1]; Z = DFT_N(z); X[k] = E[k] + W_2N^k O[k] with
// E = (Z[k] + conj Z[N-k]) / 2, O = (Z[k] - conj Z[N-k]) / (2i).
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2N, bool ZP>
__global__ void __launch_bounds__(kThreads)
fftx_fwd_kernel(const T* __restrict__ in, HFFT_C* __restrict__ out_main, HFFT_C* __restrict__ out_nyq,
                int nrows, int rows_per_cta, int rows_per_plane, int nz, int use_ms, MsParam<T> ms,
                const HFFT_C* __restrict__ tw /* exp(-2 pi i t / 2N), 2N entries */) {
    typedef HFFT_C C;
    constexpr int N = 1 << LOG2N;
    constexpr int S4 = LOG2N / 2;
    constexpr bool HAS2 = (LOG2N & 1) != 0;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int row0 = blockIdx.x * rows_per_cta;
    const int nr = min(rows_per_cta, nrows - row0);
    const long long in_rs = ZP ? N : 2 * N;   // reals per input row

    if (S4 == 0) {   // N == 2: a single radix-2 butterfly per row
        for (int r = tid; r < nr; r += kThreads) {
            const C* zin = reinterpret_cast<const C*>(in + (long long)(row0 + r) * in_rs);
            C a0 = zin[0], a1 = ZP ? mk<T>(0, 0) : zin[1];
            if (use_ms) { T sc = ms.v[((row0 + r) / rows_per_plane) % nz]; a0.x *= sc; a0.y *= sc; }
            s[r * N + 0] = cadd(a0, a1);
            s[r * N + 1] = csub(a0, a1);
        }
    } else {
        constexpr int Q0 = N / 4 > 0 ? N / 4 : 1;
        constexpr int LQ0 = LOG2N >= 2 ? LOG2N - 2 : 0;
        for (int w = tid; w < nr * Q0; w += kThreads) {
            const int r = w >> LQ0, j = w & (Q0 - 1);
            const C* zin = reinterpret_cast<const C*>(in + (long long)(row0 + r) * in_rs);
            C a0 = zin[j], a1 = zin[j + Q0], a2, a3;
            if (ZP) {
                if (use_ms) {
                    T sc = ms.v[((row0 + r) / rows_per_plane) % nz];
                    a0.x *= sc; a0.y *= sc; a1.x *= sc; a1.y *= sc;
                }
                // a2 = a3 = 0: the radix-4 butterfly degenerates
                C m1 = mul_mi(a1);
                a2 = csub(a0, a1);
                a3 = csub(a0, m1);
                C y1 = cadd(a0, m1);
                a0 = cadd(a0, a1);
                a1 = y1;
            } else {
                a2 = zin[j + 2 * Q0];
                a3 = zin[j + 3 * Q0];
                bfly4_fwd(a0, a1, a2, a3);
            }
            if (Q0 > 1) {   // W_N^{jm} = tw[2 j m]
                a1 = cmul(a1, ldtw(tw, 2 * j));
                a2 = cmul(a2, ldtw(tw, 4 * j));
                a3 = cmul(a3, ldtw(tw, 6 * j));
            }
            C* sr = s + r * N;
            sr[j] = a0; sr[j + Q0] = a1; sr[j + 2 * Q0] = a2; sr[j + 3 * Q0] = a3;
        }
        __syncthreads();
#pragma unroll
        for (int st = 1; st < S4; ++st) {
            const int log2Q = LOG2N - 2 * st - 2;
            for (int w = tid; w < nr * Q0; w += kThreads)
                dif4_stage(s + (w >> LQ0) * N, 1, w & (Q0 - 1), log2Q, tw, 2 << (2 * st));
            __syncthreads();
        }
        if (HAS2) {
            for (int w = tid; w < nr * (N / 2); w += kThreads)
                r2_stage(s + (w / (N / 2)) * N, 1, w % (N / 2));
        }
    }
    __syncthreads();

    // post-process: pairs (k, N-k), k = 0..N/2
    constexpr int NP = N / 2 + 1;
    for (int w = tid; w < nr * NP; w += kThreads) {
        const int r = w / NP, k = w - r * NP;
        const C* sr = s + r * N;
        const long long row = row0 + r;
        if (k == 0) {
            C z0 = sr[0];
            out_main[row * N] = mk<T>(z0.x + z0.y, 0);
            out_nyq[row] = mk<T>(z0.x - z0.y, 0);
        } else {
            C zk = sr[freq2pos<LOG2N>(k)], zn = sr[freq2pos<LOG2N>(N - k)];
            C E = mk<T>((zk.x + zn.x) * (T)0.5, (zk.y - zn.y) * (T)0.5);
            C O = mk<T>((zk.y + zn.y) * (T)0.5, (zn.x - zk.x) * (T)0.5);
            C WO = cmul(ldtw(tw, k), O);
            out_main[row * N + k] = cadd(E, WO);
            if (k != N - k) out_main[row * N + (N - k)] = cconj(csub(E, WO));
        }
    }
}

// ------------------------------------------------------------------------------------------
// S5: inverse x (complex-to-real, crop to the first N reals = first N/2 complex outputs).
// Z~[k] = E~ + i O~,  E~ = X[k] + conj X[N-k],  O~ = (X[k] - conj X[N-k]) W_2N^{-k};
// z~ = IDFT_N(Z~) holds x~[2t] + i x~[2t+1].
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2N>
__global__ void __launch_bounds__(kThreads)
ifftx_kernel(const HFFT_C* __restrict__ in_main, const HFFT_C* __restrict__ in_nyq, T* __restrict__ out,
             int nrows, int rows_per_cta, const HFFT_C* __restrict__ tw) {
    typedef HFFT_C C;
    constexpr int N = 1 << LOG2N;
    constexpr int S4 = LOG2N / 2;
    constexpr bool HAS2 = (LOG2N & 1) != 0;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int row0 = blockIdx.x * rows_per_cta;
    const int nr = min(rows_per_cta, nrows - row0);

    constexpr int NP = N / 2 + 1;
    for (int w = tid; w < nr * NP; w += kThreads) {
        const int r = w / NP, k = w - r * NP;
        C* sr = s + r * N;
        const long long row = row0 + r;
        C xk = in_main[row * N + k];    // k <= N/2 < N
        C xn = (k == 0) ? in_nyq[row] : in_main[row * N + (N - k)];
        C E = mk<T>(xk.x + xn.x, xk.y - xn.y);
        C D = mk<T>(xk.x - xn.x, xk.y + xn.y);
        C O = (k == 0) ? D : cmulc(D, ldtw(tw, k));
        // Z~[k] = E + i O ; Z~[N-k] = conj(E) + i conj(O)
        sr[freq2pos<LOG2N>(k)] = mk<T>(E.x - O.y, E.y + O.x);
        if (k != 0 && k != N - k) sr[freq2pos<LOG2N>(N - k)] = mk<T>(E.x + O.y, O.x - E.y);
    }
    __syncthreads();

    if (S4 == 0) {   // N == 2: z~[0] = Z~[0] + Z~[1]
        for (int r = tid; r < nr; r += kThreads) {
            C v = cadd(s[r * N], s[r * N + 1]);
            *reinterpret_cast<C*>(out + (long long)(row0 + r) * N) = v;
        }
        return;
    }
    constexpr int Q0 = N / 4 > 0 ? N / 4 : 1;
    constexpr int LQ0 = LOG2N >= 2 ? LOG2N - 2 : 0;
    if (HAS2) {
        for (int w = tid; w < nr * (N / 2); w += kThreads)
            r2_stage(s + (w / (N / 2)) * N, 1, w % (N / 2));
        __syncthreads();
    }
#pragma unroll
    for (int st = S4 - 1; st >= 1; --st) {   // block length L = N >> 2 st, growing
        const int log2Q = LOG2N - 2 * st - 2;
        for (int w = tid; w < nr * Q0; w += kThreads)
            dit4_stage(s + (w >> LQ0) * N, 1, w & (Q0 - 1), log2Q, tw, 2 << (2 * st));
        __syncthreads();
    }
    // last stage (L = N) fused with the cropped store
    for (int w = tid; w < nr * Q0; w += kThreads) {
        const int r = w >> LQ0, j = w & (Q0 - 1);
        const C* sr = s + r * N;
        C b0 = sr[j], b1 = sr[j + Q0], b2 = sr[j + 2 * Q0], b3 = sr[j + 3 * Q0];
        if (Q0 > 1) {
            b1 = cmulc(b1, ldtw(tw, 2 * j));
            b2 = cmulc(b2, ldtw(tw, 4 * j));
            b3 = cmulc(b3, ldtw(tw, 6 * j));
        }
        C t0 = cadd(b0, b2), t1 = csub(b0, b2), t2 = cadd(b1, b3), t3 = csub(b1, b3);
        C* zout = reinterpret_cast<C*>(out + (long long)(row0 + r) * N);
        zout[j] = cadd(t0, t2);
        zout[j + Q0] = cadd(t1, mul_pi(t3));
    }
}

// ------------------------------------------------------------------------------------------
// S2 / S4: transforms along y on groups of G adjacent kx columns (main blocks), and on the
// Nyquist column of G planes at a time (tail blocks).  Shared layout s[e * G + g].
// ------------------------------------------------------------------------------------------
struct YGeom {
    int nblk_main;        // blocks handling main columns
    int groups_per_plane; // ceil(nx / G)
    int G;
    int nx;
    int nplanes;
    int nz;               // for the i-rotation of z planes (0: no rotation)
    int rows;             // rows per plane on the row side (ny on the hot path, 2ny for the bank)
    long long row_nyq_off;   // offset of the Nyquist array on the row side = nplanes * rows * nx
    long long k_plane_stride;   // KS
};

struct YAddr {
    long long row_base, k_base;
    long long row_gs, k_gs;   // stride between the G sequences
    long long row_es, k_es;   // stride between consecutive elements of one sequence
    int gcount, plane0, plane_gs;
};

__device__ __forceinline__ YAddr y_addr(const YGeom& g, int N) {
    YAddr a;
    int b = blockIdx.x;
    if (b < g.nblk_main) {
        int p = b / g.groups_per_plane, g0 = (b - p * g.groups_per_plane) * g.G;
        a.row_base = (long long)p * g.rows * g.nx + g0;
        a.k_base = (long long)p * g.k_plane_stride + g0;
        a.row_gs = 1; a.k_gs = 1; a.row_es = g.nx; a.k_es = g.nx;
        a.gcount = min(g.G, g.nx - g0);
        a.plane0 = p; a.plane_gs = 0;
    } else {
        int p0 = (b - g.nblk_main) * g.G;
        a.row_base = g.row_nyq_off + (long long)p0 * g.rows;
        a.k_base = (long long)p0 * g.k_plane_stride + (long long)N * g.nx;
        a.row_gs = g.rows; a.k_gs = g.k_plane_stride; a.row_es = 1; a.k_es = 1;
        a.gcount = min(g.G, g.nplanes - p0);
        a.plane0 = p0; a.plane_gs = 1;
    }
    return a;
}

template <typename T, int LOG2N, bool ZP>
__global__ void __launch_bounds__(kThreads)
ffty_fwd_kernel(const HFFT_C* __restrict__ in, HFFT_C* __restrict__ out, YGeom geo,
                const HFFT_C* __restrict__ tw /* N entries */) {
    typedef HFFT_C C;
    constexpr int N = 1 << LOG2N;
    constexpr int S4 = LOG2N / 2;
    constexpr bool HAS2 = (LOG2N & 1) != 0;
    constexpr int Q0 = N / 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int G = geo.G;
    const YAddr ad = y_addr(geo, N);

    for (int w = tid; w < G * Q0; w += kThreads) {
        const int j = w / G, g = w - j * G;
        if (g >= ad.gcount) continue;
        const C* src = in + ad.row_base + g * ad.row_gs;
        C a0 = src[(long long)j * ad.row_es], a1 = src[(long long)(j + Q0) * ad.row_es], a2, a3;
        if (ZP) {
            C m1 = mul_mi(a1);
            a2 = csub(a0, a1);
            a3 = csub(a0, m1);
            C y1 = cadd(a0, m1);
            a0 = cadd(a0, a1);
            a1 = y1;
        } else {
            a2 = src[(long long)(j + 2 * Q0) * ad.row_es];
            a3 = src[(long long)(j + 3 * Q0) * ad.row_es];
            bfly4_fwd(a0, a1, a2, a3);
        }
        if (Q0 > 1) {
            a1 = cmul(a1, ldtw(tw, j));
            a2 = cmul(a2, ldtw(tw, 2 * j));
            a3 = cmul(a3, ldtw(tw, 3 * j));
        }
        s[(j)*G + g] = a0; s[(j + Q0) * G + g] = a1; s[(j + 2 * Q0) * G + g] = a2; s[(j + 3 * Q0) * G + g] = a3;
    }
    __syncthreads();
#pragma unroll
    for (int st = 1; st < S4; ++st) {
        const int log2Q = LOG2N - 2 * st - 2;
        for (int w = tid; w < G * Q0; w += kThreads) {
            const int t = w / G, g = w - t * G;
            dif4_stage(s + g, G, t, log2Q, tw, 1 << (2 * st));
        }
        __syncthreads();
    }
    if (HAS2) {
        for (int w = tid; w < G * (N / 2); w += kThreads) {
            const int t = w / G, g = w - t * G;
            r2_stage(s + g, G, t);
        }
        __syncthreads();
    }
    for (int w = tid; w < G * N; w += kThreads) {
        const int p = w / G, g = w - p * G;
        if (g >= ad.gcount) continue;
        C v = s[p * G + g];
        if (geo.nz > 0) {
            int plane = ad.plane0 + g * ad.plane_gs;
            if ((plane / geo.nz) % 3 == 2) v = mul_pi(v);   // M'_z = i M_z
        }
        out[ad.k_base + g * ad.k_gs + (long long)pos2freq<LOG2N>(p) * ad.k_es] = v;
    }
}

template <typename T, int LOG2N>
__global__ void __launch_bounds__(kThreads)
iffty_kernel(const HFFT_C* __restrict__ in, HFFT_C* __restrict__ out, YGeom geo, const HFFT_C* __restrict__ tw) {
    typedef HFFT_C C;
    constexpr int N = 1 << LOG2N;
    constexpr int S4 = LOG2N / 2;
    constexpr bool HAS2 = (LOG2N & 1) != 0;
    constexpr int Q0 = N / 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int G = geo.G;
    const YAddr ad = y_addr(geo, N);

    for (int w = tid; w < G * N; w += kThreads) {
        const int k = w / G, g = w - k * G;
        if (g >= ad.gcount) continue;
        C v = in[ad.k_base + g * ad.k_gs + (long long)k * ad.k_es];
        if (geo.nz > 0) {
            int plane = ad.plane0 + g * ad.plane_gs;
            if ((plane / geo.nz) % 3 == 2) v = mul_mi(v);   // H_z = -i H'_z
        }
        s[freq2pos<LOG2N>(k) * G + g] = v;
    }
    __syncthreads();
    if (HAS2) {
        for (int w = tid; w < G * (N / 2); w += kThreads) {
            const int t = w / G, g = w - t * G;
            r2_stage(s + g, G, t);
        }
        __syncthreads();
    }
#pragma unroll
    for (int st = S4 - 1; st >= 1; --st) {
        const int log2Q = LOG2N - 2 * st - 2;
        for (int w = tid; w < G * Q0; w += kThreads) {
            const int t = w / G, g = w - t * G;
            dit4_stage(s + g, G, t, log2Q, tw, 1 << (2 * st));
        }
        __syncthreads();
    }
    for (int w = tid; w < G * Q0; w += kThreads) {
        const int j = w / G, g = w - j * G;
        if (g >= ad.gcount) continue;
        C b0 = s[(j)*G + g], b1 = s[(j + Q0) * G + g], b2 = s[(j + 2 * Q0) * G + g], b3 = s[(j + 3 * Q0) * G + g];
        if (Q0 > 1) {
            b1 = cmulc(b1, ldtw(tw, j));
            b2 = cmulc(b2, ldtw(tw, 2 * j));
            b3 = cmulc(b3, ldtw(tw, 3 * j));
        }
        C t0 = cadd(b0, b2), t1 = csub(b0, b2), t2 = cadd(b1, b3), t3 = csub(b1, b3);
        C* dst = out + ad.row_base + g * ad.row_gs;
        dst[(long long)j * ad.row_es] = cadd(t0, t2);
        dst[(long long)(j + Q0) * ad.row_es] = cadd(t1, mul_pi(t3));
    }
}

// ------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------
template <typename T> static int x_rows_per_cta(int N) {
    int elems = 2048;
    int r = elems / N;
    return r < 1 ? 1 : r;
}
template <typename T> static int y_group(int nx) {
    int G = (int)(64 / sizeof(HFFT_C));   // 64-byte segments: 8 (f32) or 4 (f64) columns
    return nx < G ? nx : G;
}

// opt in to > 48 KB of dynamic shared memory once per kernel instantiation (`done` is a static
// local of the dispatch case, i.e. one flag per instantiation)
template <typename K> static cudaError_t set_smem(K kernel, size_t bytes, size_t& done) {
    if (bytes <= 48 * 1024 || bytes <= done) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) done = bytes;
    return e;
}

#define HFFT_DISPATCH_LOG2(LG, LO, HI, ...)                                                        \
    switch (LG) {                                                                                   \
        case 1: { constexpr int L = (1 < LO) ? LO : ((1 > HI) ? HI : 1); if (L == 1) { __VA_ARGS__ } break; }   \
        case 2: { constexpr int L = (2 < LO) ? LO : ((2 > HI) ? HI : 2); if (L == 2) { __VA_ARGS__ } break; }   \
        case 3: { constexpr int L = (3 < LO) ? LO : ((3 > HI) ? HI : 3); if (L == 3) { __VA_ARGS__ } break; }   \
        case 4: { constexpr int L = (4 < LO) ? LO : ((4 > HI) ? HI : 4); if (L == 4) { __VA_ARGS__ } break; }   \
        case 5: { constexpr int L = (5 < LO) ? LO : ((5 > HI) ? HI : 5); if (L == 5) { __VA_ARGS__ } break; }   \
        case 6: { constexpr int L = (6 < LO) ? LO : ((6 > HI) ? HI : 6); if (L == 6) { __VA_ARGS__ } break; }   \
        case 7: { constexpr int L = (7 < LO) ? LO : ((7 > HI) ? HI : 7); if (L == 7) { __VA_ARGS__ } break; }   \
        case 8: { constexpr int L = (8 < LO) ? LO : ((8 > HI) ? HI : 8); if (L == 8) { __VA_ARGS__ } break; }   \
        case 9: { constexpr int L = (9 < LO) ? LO : ((9 > HI) ? HI : 9); if (L == 9) { __VA_ARGS__ } break; }   \
        case 10: { constexpr int L = (10 < LO) ? LO : ((10 > HI) ? HI : 10); if (L == 10) { __VA_ARGS__ } break; } \
        case 11: { constexpr int L = (11 < LO) ? LO : ((11 > HI) ? HI : 11); if (L == 11) { __VA_ARGS__ } break; } \
        default: break;                                                                             \
    }

template <typename T, bool ZP>
cudaError_t launch_fftx_fwd(const T* in, void* out_main, void* out_nyq, int log2nx, int nrows, int rows_per_plane,
                            int nz, const double* ms_host, const void* tw, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2nx;
    const int rpc = x_rows_per_cta<T>(N);
    const size_t smem = (size_t)rpc * N * sizeof(C);
    const int grid = (nrows + rpc - 1) / rpc;
    MsParam<T> ms;
    const int use_ms = ms_host != nullptr;
    for (int k = 0; k < HFFT_MAX_NZ; ++k) ms.v[k] = (use_ms && k < nz) ? (T)ms_host[k] : (T)1;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_LOG2(log2nx, 1, 10, {
        auto kern = fftx_fwd_kernel<T, L, ZP>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<grid, kThreads, smem, st>>>(in, (C*)out_main, (C*)out_nyq, nrows, rpc, rows_per_plane,
                                               nz > 0 ? nz : 1, use_ms, ms, (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_ifftx(const void* in_main, const void* in_nyq, T* out, int log2nx, int nrows, const void* tw,
                         cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2nx;
    const int rpc = x_rows_per_cta<T>(N);
    const size_t smem = (size_t)rpc * N * sizeof(C);
    const int grid = (nrows + rpc - 1) / rpc;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_LOG2(log2nx, 1, 10, {
        auto kern = ifftx_kernel<T, L>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<grid, kThreads, smem, st>>>((const C*)in_main, (const C*)in_nyq, out, nrows, rpc, (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

template <typename T>
static YGeom make_ygeom(int nx, int log2N, int nplanes, int nz_rot, int rows, long long ks) {
    YGeom g;
    g.G = y_group<T>(nx);
    g.nx = nx;
    g.groups_per_plane = (nx + g.G - 1) / g.G;
    g.nblk_main = g.groups_per_plane * nplanes;
    g.nplanes = nplanes;
    g.nz = nz_rot;
    g.rows = rows;
    g.row_nyq_off = (long long)nplanes * rows * nx;
    g.k_plane_stride = ks;
    (void)log2N;
    return g;
}

template <typename T, bool ZP>
cudaError_t launch_ffty_fwd(const void* in, void* out, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                            const void* tw, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2N;
    YGeom g = make_ygeom<T>(nx, log2N, nplanes, nz_rot, ZP ? N / 2 : N, ks);
    const size_t smem = (size_t)g.G * N * sizeof(C);
    const int grid = g.nblk_main + (nplanes + g.G - 1) / g.G;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_LOG2(log2N, 2, 11, {
        auto kern = ffty_fwd_kernel<T, L, ZP>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<grid, kThreads, smem, st>>>((const C*)in, (C*)out, g, (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_iffty(const void* in, void* out, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                         const void* tw, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2N;
    YGeom g = make_ygeom<T>(nx, log2N, nplanes, nz_rot, N / 2, ks);
    const size_t smem = (size_t)g.G * N * sizeof(C);
    const int grid = g.nblk_main + (nplanes + g.G - 1) / g.G;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_LOG2(log2N, 2, 11, {
        auto kern = iffty_kernel<T, L>;
        static size_t smem_done = 0;
        err = set_smem(kern, smem, smem_done);
        if (err == cudaSuccess) {
            kern<<<grid, kThreads, smem, st>>>((const C*)in, (C*)out, g, (const C*)tw);
            err = cudaGetLastError();
        }
    })
    return err;
}

// explicit instantiations used by hfft_api.cu / tensor_build.cu
template cudaError_t launch_fftx_fwd<float, true>(const float*, void*, void*, int, int, int, int, const double*, const void*, cudaStream_t);
template cudaError_t launch_fftx_fwd<double, true>(const double*, void*, void*, int, int, int, int, const double*, const void*, cudaStream_t);
template cudaError_t launch_fftx_fwd<double, false>(const double*, void*, void*, int, int, int, int, const double*, const void*, cudaStream_t);
template cudaError_t launch_ifftx<float>(const void*, const void*, float*, int, int, const void*, cudaStream_t);
template cudaError_t launch_ifftx<double>(const void*, const void*, double*, int, int, const void*, cudaStream_t);
template cudaError_t launch_ffty_fwd<float, true>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_ffty_fwd<double, true>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_ffty_fwd<double, false>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_iffty<float>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);
template cudaError_t launch_iffty<double>(const void*, void*, int, int, int, int, long long, const void*, cudaStream_t);

}  // namespace hfft
