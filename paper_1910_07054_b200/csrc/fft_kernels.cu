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
//   M^ (after S2)   [plane][KS] C, element k = kx * 2ny + ky; "mirror" layout: kx * (2ny + 2) + ypos(ky), where
//                   ypos pairs ky with 2ny - ky in adjacent slots (see ypos below)
// The z-component planes of M^ hold i*M_z (and H^ holds i*H_z) so that the layer coupling is a
// real matrix acting on real and imaginary parts alike.
//
// All four kernels are PERSISTENT: a CTA walks a contiguous chunk of rows (row blocks), so that
// everything that depends on the thread only -- twiddles, swizzled shared-memory addresses --
// is set up once (RowFFT::Ctx, fft.cuh), and the global loads of the next row are issued
// before the butterflies of the current one.
#include "hfft_internal.h"
#include "fft.cuh"

namespace hfft {

// CTA size limit of the x kernels (fp32: 2 CTAs of 512 per SM, i.e. at most 64 registers per thread)
// (a 1024-thread CTA with 16 rows per block -- 128-byte instead of 64-byte runs of X^ at nx = 512 -- measured the same:
// B200, C5, S1 0.632 vs 0.638 ms)
template <typename T> struct XCfg {
    static constexpr int MAXT = sizeof(T) == 4 ? 512 : 256;
    static constexpr int MINB = sizeof(T) == 4 ? 2 : 1;
};

// first shared-space address >= the dynamic shared memory base that is a multiple of `align`
__device__ __forceinline__ unsigned smem_base_aligned(unsigned align) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    return (smem_u32(smem_raw) + align - 1) & ~(align - 1);
}

// Element-index XOR of row r in a block of 2^log2rb rows (x kernels).  The transposed phase reads
// one element index from 2^log2rb rows at a time, lanes along the rows: spreading r over bits
// 0..3 of the index makes those rows hit different banks (r itself for 16 rows, 2r for 8, ...).
__device__ __forceinline__ int row_xor(int r, int log2rb, int N) {
    const int sh = log2rb < 4 ? 4 - log2rb : 0;
    return (r << sh) & 15 & (N - 1);
}

// ------------------------------------------------------------------------------------------
// S1: forward x.  A real row of 2N samples (only the first N non-zero if ZP) is packed as N
// complex z[t] = x[2t] + i x[2t+1]; Z = DFT_N(z); X[k] = E[k] + W_2N^k O[k] with
// E = (Z[k] + conj Z[N-k]) / 2, O = (Z[k] - conj Z[N-k]) / (2i).
// One row block = rb consecutive rows (y) of one plane.  Phase 1: thread (r, j) transforms row r.
// Phase 2: thread (kk, rr) forms the pairs X[k], X[N-k], k = kk + TPR it, of row rr -- lanes run
// along y so that every store to the transposed X^ is a run of rb consecutive elements.  The
// element index of row r is XOR-ed with r in shared memory, which makes the phase-2 reads
// (same k, 16 different rows) conflict free.
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2N, bool ZP>
__global__ void __launch_bounds__(XCfg<T>::MAXT, XCfg<T>::MINB)
fftx_fwd_kernel(const T* __restrict__ in, HFFT_C* __restrict__ xhat, int log2rb, int rows_per_plane, int nz,
                int use_ms, MsParam<T> ms, const HFFT_C* __restrict__ tw /* exp(-2 pi i t / 2N), 2N entries */,
                const HFFT_C* __restrict__ twt, long long nblocks, int bpc) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, false, ZP, false> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR, SH = F::SH;
    constexpr int RL = (ZP && R > 1) ? R / 2 : R;            // loads per thread
    constexpr int IT = R > 1 ? R / 2 : 1;                    // phase-2 iterations: k = kk + TPR it < N / 2
    constexpr int PZ = F::EXCH & 1;                          // buffer that receives Z (the next free one)
    const int tid = threadIdx.x, rb = 1 << log2rb;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);    // phase 1
    const int rr = tid & (rb - 1), kk = tid >> log2rb;       // phase 2
    const unsigned base = smem_base_aligned(F::ROW_BYTES);
    typename F::Ctx c;
    F::init(c, r, base + r * F::ROW_BYTES, j, row_xor(r, log2rb, N), twt, rb > 15 ? 2 : 1);
    const unsigned zrow = (base + rr * F::ROW_BYTES) ^ ((unsigned)row_xor(rr, log2rb, N) << SH) ^ (PZ ? F::BUF_BYTES : 0u);

    long long blk = (long long)blockIdx.x * bpc;
    const int nit = (int)((nblocks - blk < bpc) ? nblocks - blk : bpc);
    const int bpp = rows_per_plane >> log2rb;                // row blocks per plane
    long long plane = blk / bpp;
    int y0 = (int)(blk - plane * bpp) << log2rb;
    int layer = (int)(plane % nz);
    const C* zin = reinterpret_cast<const C*>(in) + (blk * rb + r) * (ZP ? N / 2 : N) + j;
    const long long zstep = (long long)rb * (ZP ? N / 2 : N);
    C v[R];
    pdl_wait();                                              // the previous kernel of the stream may still write `in`
#pragma unroll
    for (int q = 0; q < RL; ++q) v[q] = zin[q * TPR];

    for (int it0 = 0; it0 < nit; ++it0) {
        if (ZP && use_ms) {
            const T sc = ms.v[layer];
#pragma unroll
            for (int q = 0; q < RL; ++q) v[q] = cscale(sc, v[q]);
        }
        F::run(v, c);
#pragma unroll
        for (int q = 0; q < R; ++q) sts(F::template elem_addr<PZ>(c, q), v[q]);
        if (it0 + 1 < nit) {                                 // next block's loads fly during phase 2
            zin += zstep;
#pragma unroll
            for (int q = 0; q < RL; ++q) v[q] = zin[q * TPR];
        }
        __syncthreads();

        C* xp = xhat + plane * (long long)(N + 1) * rows_per_plane + y0 + rr;
#pragma unroll
        for (int it = 0; it < IT; ++it) {
            const int k = kk + TPR * it;
            if (it == 0 && kk == 0) {
                const C z0 = lds<C>(zrow);
                xp[0] = mk<T>(z0.x + z0.y, 0);
                xp[(long long)N * rows_per_plane] = mk<T>(z0.x - z0.y, 0);
                const C zm = lds<C>(zrow ^ ((unsigned)swz(N / 2) << SH));
                xp[(long long)(N / 2) * rows_per_plane] = cconj(zm);           // W_2N^{N/2} = -i
            } else {
                const C zk = lds<C>(zrow ^ ((unsigned)swz(k) << SH));
                const C zn = cconj(lds<C>(zrow ^ ((unsigned)swz(N - k) << SH)));
                const C s = cadd(zk, zn);                                      // 2 E
                const C wo = cmul(mul_mi(csub(zk, zn)), __ldg(tw + k));        // 2 W O
                xp[(long long)k * rows_per_plane] = cscale((T)0.5, cadd(s, wo));
                xp[(long long)(N - k) * rows_per_plane] = cconj(cscale((T)0.5, csub(s, wo)));
            }
        }
        __syncthreads();                                     // Z is consumed before the next block's exchanges
        y0 += rb;
        if (y0 == rows_per_plane) { y0 = 0; ++plane; if (++layer == nz) layer = 0; }
    }
}

// ------------------------------------------------------------------------------------------
// S5: inverse x (complex-to-real, crop to the first N reals = first N/2 complex outputs).
// Z~[k] = E~ + i O~,  E~ = X[k] + conj X[N-k],  O~ = (X[k] - conj X[N-k]) W_2N^{-k};
// z~ = IDFT_N(Z~) holds x~[2t] + i x~[2t+1].  Same row blocks as S1: the block's tile of the
// transposed X^ ([N + 1][rb]) is brought to shared memory by cp.async ONE BLOCK AHEAD (ncu: without
// it the kernel waits on the global loads, long_scoreboard 7.2 + barrier 3.6 per issue); phase 1
// reads it with lanes along y and writes Z~ to the rows, phase 2 is the row transform; only the
// first half of its outputs is stored (fused crop).
// ------------------------------------------------------------------------------------------
// RED (hfft_plan_set_reduction): the epilogue also accumulates, per plane, the sum of h
// and the sum of m h over the plane's cells (doubles, one atomicAdd per warp and block) into
// sums[plane][2] -- the layer average <H_z> of PAPER.md:209 and the m.H sums of the demagnetization energy.
template <typename T, int LOG2N, bool RED>
__global__ void __launch_bounds__(XCfg<T>::MAXT, 1)
ifftx_kernel(const HFFT_C* __restrict__ xhat, T* __restrict__ out, int log2rb, int rows_per_plane,
             const HFFT_C* __restrict__ tw, const HFFT_C* __restrict__ twt, long long nblocks, int bpc,
             const T* __restrict__ m, double* __restrict__ sums) {
    typedef HFFT_C C;
    // fp32: twiddles in registers and one 512-thread CTA per SM (112-122 registers) -- measured against table twiddles
    // with two CTAs per SM (64 registers): C5 S5 0.712 -> 0.672 ms, C3 0.0178 -> 0.0167 ms, C4 0.0516 -> 0.0505 ms; the
    // same change does nothing for S1 (C5 0.700 -> 0.716 ms), which keeps the table
    typedef RowFFT<T, LOG2N, true, false, sizeof(T) == 4> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR, SH = F::SH;
    constexpr int IT = R > 1 ? R / 2 : 1;
    constexpr int RS = R > 1 ? R / 2 : 1;                    // stores per thread (crop)
    constexpr int PZ = 1;                                    // Z~ sits in buffer 1: exchange 0 writes buffer 0
    const int tid = threadIdx.x, rb = 1 << log2rb, nthreads = blockDim.x;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);    // phase 2
    const int rr = tid & (rb - 1), kk = tid >> log2rb;       // phase 1
    const unsigned base = smem_base_aligned(F::ROW_BYTES);
    typename F::Ctx c;
    F::init(c, r, base + r * F::ROW_BYTES, j, row_xor(r, log2rb, N), twt, rb > 15 ? 2 : 1);
    const unsigned zrow = (base + rr * F::ROW_BYTES) ^ ((unsigned)row_xor(rr, log2rb, N) << SH) ^ F::BUF_BYTES;
    // staging tile of the block's X^ values, [N + 1][rb], filled by cp.async one block ahead
    const unsigned stg = base + rb * F::ROW_BYTES;
    const int log2cpr = log2rb + SH - 4;                     // 16-byte chunks per kx row of the tile
    const int nchunks = (N + 1) << log2cpr;

    long long blk = (long long)blockIdx.x * bpc;
    const int nit = (int)((nblocks - blk < bpc) ? nblocks - blk : bpc);
    const int bpp = rows_per_plane >> log2rb;
    long long plane = blk / bpp;
    int y0 = (int)(blk - plane * bpp) << log2rb;
    C* zout = reinterpret_cast<C*>(out) + (blk * rb + r) * (N / 2) + j;
    const C* zm = reinterpret_cast<const C*>(m) + (blk * rb + r) * (N / 2) + j;
    const long long zstep = (long long)rb * (N / 2);

    auto fetch = [&](long long pl, int yy) {
        const char* src = reinterpret_cast<const char*>(xhat + pl * (long long)(N + 1) * rows_per_plane + yy);
        for (int x = tid; x < nchunks; x += nthreads) {
            const int k = x >> log2cpr, ch = x & ((1 << log2cpr) - 1);
            cp_async16(stg + ((unsigned)x << 4), src + ((long long)k * rows_per_plane * sizeof(C) + ((long long)ch << 4)));
        }
        cp_async_commit();
    };
    pdl_wait();                                              // X^ comes from the previous kernel (S4)
    fetch(plane, y0);

    for (int it0 = 0; it0 < nit; ++it0) {
        cp_async_wait_group<0>();
        __syncthreads();                                     // the tile has landed for every thread
        const unsigned sx = stg + ((unsigned)rr << SH);
        const unsigned kstride = (unsigned)rb << SH;
#pragma unroll
        for (int it = 0; it < IT; ++it) {
            const int k = kk + TPR * it;
            if (it == 0 && kk == 0) {
                const C x0 = lds<C>(sx), xn = lds<C>(sx + N * kstride);            // DC and Nyquist (both real)
                const C e = cadd(x0, cconj(xn)), d = csub(x0, cconj(xn));
                sts(zrow, mk<T>(e.x - d.y, e.y + d.x));
                const C xm = lds<C>(sx + (N / 2) * kstride);
                sts(zrow ^ ((unsigned)swz(N / 2) << SH), mk<T>(2 * xm.x, -2 * xm.y));
            } else {
                const C xk = lds<C>(sx + k * kstride);
                const C xn = cconj(lds<C>(sx + (N - k) * kstride));
                const C e = cadd(xk, xn);
                const C o = mul_pi(cmulc(csub(xk, xn), __ldg(tw + k)));        // i O~
                sts(zrow ^ ((unsigned)swz(k) << SH), cadd(e, o));              // Z~[k] = E~ + i O~
                sts(zrow ^ ((unsigned)swz(N - k) << SH), cconj(csub(e, o)));   // Z~[N-k] = conj(E~ - i O~)
            }
        }
        __syncthreads();                                     // Z~ complete; the staging tile is free
        const long long cur_plane = plane;
        y0 += rb;
        if (y0 == rows_per_plane) { y0 = 0; ++plane; }
        if (it0 + 1 < nit) fetch(plane, y0);                 // next block's tile flies during the transform
        C v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = lds<C>(F::template elem_addr<PZ>(c, q));
        F::run(v, c);
#pragma unroll
        for (int q = 0; q < RS; ++q) zout[q * TPR] = v[q];
        if constexpr (RED) {
            double sh = 0.0, smh = 0.0;
#pragma unroll
            for (int q = 0; q < RS; ++q) {
                const C mm = zm[q * TPR];
                sh += (double)v[q].x + (double)v[q].y;
                smh += (double)v[q].x * (double)mm.x + (double)v[q].y * (double)mm.y;
            }
            if (nthreads >= 32) {                            // a block lies in one plane: so does the warp
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    sh += __shfl_xor_sync(0xffffffffu, sh, o);
                    smh += __shfl_xor_sync(0xffffffffu, smh, o);
                }
            }
            if (nthreads < 32 || (tid & 31) == 0) {
                atomicAdd(sums + 2 * cur_plane, sh);
                atomicAdd(sums + 2 * cur_plane + 1, smh);
            }
            zm += zstep;
        }
        zout += zstep;
    }
}

// ------------------------------------------------------------------------------------------
// S2 / S4: transforms along y on the contiguous rows of the transposed X^.  Row = (plane, kx);
// a CTA holds blockDim / TPR rows at a time and walks `gpc` consecutive row groups.
// ------------------------------------------------------------------------------------------
template <int LOG2N> struct YCfg {
    static constexpr int TPR = (1 << LOG2N) / (LOG2N < 3 ? (1 << LOG2N) : 8);
    static constexpr int THREADS = TPR > 128 ? TPR : 128;
};

// Mirror layout of a spectrum row (hfft_plan_set_mirror): the tensor spectra are even (xx, yy, zz, xz) or
// odd (xy, yz) in ky, so ky and 2ny - ky can share one bank entry.  A row then has N + 2 slots: ky <= N/2 sits at
// 2 ky, its mirror N - ky at 2 ky + 1; ky = 0 and ky = N/2 are their own mirrors, their odd slots (1 and N + 1) are
// dummies that hold zeros (never written by S2, H^ = N^ 0 = 0 written by S3, ignored by S4).
__device__ __forceinline__ int ypos(int ky, int N, int mirror) {
    return mirror ? (ky <= N / 2 ? 2 * ky : 2 * (N - ky) + 1) : ky;
}

// (plane, kx) of a row and whether the plane is a z component (nz_rot layers per component)
struct RowPos {
    long long plane; int kx; int pl3;
    __device__ __forceinline__ void set(long long row, int nxp1, int nz_rot) {
        plane = row / nxp1; kx = (int)(row - plane * nxp1);
        pl3 = nz_rot > 0 ? (int)(plane % (3 * nz_rot)) : 0;
    }
    __device__ __forceinline__ void advance(int rows, int nxp1, int nz_rot) {
        kx += rows;
        while (kx >= nxp1) { kx -= nxp1; ++plane; if (++pl3 == 3 * nz_rot) pl3 = 0; }
    }
    __device__ __forceinline__ bool is_z(int nz_rot) const { return nz_rot > 0 && pl3 >= 2 * nz_rot; }
};

template <typename T, int LOG2N, bool ZP>
__global__ void __launch_bounds__(YCfg<LOG2N>::THREADS)
ffty_fwd_kernel(const HFFT_C* __restrict__ xhat, HFFT_C* __restrict__ spec, long long nrows, int nxp1, int nz_rot,
                long long ks, const HFFT_C* __restrict__ twt, long long ngroups, int gpc, int mirror) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, false, ZP, sizeof(T) == 4> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR;
    constexpr int RL = ZP ? R / 2 : R;
    const int tid = threadIdx.x;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);
    const int rpc = blockDim.x >> F::LOG2TPR;
    typename F::Ctx c;
    F::init(c, r, smem_base_aligned(F::ROW_BYTES) + r * F::ROW_BYTES, j, 0, twt);

    const long long g0 = (long long)blockIdx.x * gpc;
    const int nit = (int)((ngroups - g0 < gpc) ? ngroups - g0 : gpc);
    long long row = g0 * rpc + r;
    RowPos pos; pos.set(row < nrows ? row : nrows - 1, nxp1, nz_rot);
    const C* zin = xhat + row * (ZP ? N / 2 : N) + j;
    const long long zstep = (long long)rpc * (ZP ? N / 2 : N);
    C nv[RL];
    bool live = row < nrows;
    pdl_wait();                                              // X^ comes from the previous kernel (S1)
    if (live) {
#pragma unroll
        for (int q = 0; q < RL; ++q) nv[q] = zin[q * TPR];
    }
    for (int it = 0; it < nit; ++it) {
        C v[R];
#pragma unroll
        for (int q = 0; q < RL; ++q) v[q] = nv[q];
        const bool cur_live = live;
        const bool rot = pos.is_z(nz_rot);
        C* dst = spec + pos.plane * ks + (long long)pos.kx * (mirror ? N + 2 : N);
        row += rpc; zin += zstep;
        live = (it + 1 < nit) && row < nrows;
        if (live) {
            pos.advance(rpc, nxp1, nz_rot);
#pragma unroll
            for (int q = 0; q < RL; ++q) nv[q] = zin[q * TPR];
        }
        F::run(v, c);
        if (cur_live) {
            if (rot) {                                       // M'_z = i M_z
#pragma unroll
                for (int q = 0; q < R; ++q) v[q] = mul_pi(v[q]);
            }
#pragma unroll
            for (int q = 0; q < R; ++q) dst[ypos(j + q * TPR, N, mirror)] = v[q];
        }
    }
}

template <typename T, int LOG2N>
__global__ void __launch_bounds__(YCfg<LOG2N>::THREADS)
iffty_kernel(const HFFT_C* __restrict__ spec, HFFT_C* __restrict__ xhat, long long nrows, int nxp1, int nz_rot,
             long long ks, const HFFT_C* __restrict__ twt, long long ngroups, int gpc, int mirror) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, true, false, sizeof(T) == 4> F;
    constexpr int N = F::N, R = F::R, TPR = F::TPR;
    const int tid = threadIdx.x;
    const int r = tid >> F::LOG2TPR, j = tid & (TPR - 1);
    const int rpc = blockDim.x >> F::LOG2TPR;
    typename F::Ctx c;
    F::init(c, r, smem_base_aligned(F::ROW_BYTES) + r * F::ROW_BYTES, j, 0, twt);

    const long long g0 = (long long)blockIdx.x * gpc;
    const int nit = (int)((ngroups - g0 < gpc) ? ngroups - g0 : gpc);
    long long row = g0 * rpc + r;
    RowPos pos; pos.set(row < nrows ? row : nrows - 1, nxp1, nz_rot);
    C nv[R];
    bool live = row < nrows;
    pdl_wait();                                              // H^ comes from the previous kernel (S3)
    if (live) {
        const C* src = spec + pos.plane * ks + (long long)pos.kx * (mirror ? N + 2 : N);
#pragma unroll
        for (int q = 0; q < R; ++q) nv[q] = src[ypos(j + q * TPR, N, mirror)];
    }
    for (int it = 0; it < nit; ++it) {
        C v[R];
        const bool cur_live = live;
        const bool rot = pos.is_z(nz_rot);
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = rot ? mul_mi(nv[q]) : nv[q];        // H_z = -i H'_z
        C* dst = xhat + row * (N / 2) + j;
        row += rpc;
        live = (it + 1 < nit) && row < nrows;
        if (live) {
            pos.advance(rpc, nxp1, nz_rot);
            const C* src = spec + pos.plane * ks + (long long)pos.kx * (mirror ? N + 2 : N);
#pragma unroll
            for (int q = 0; q < R; ++q) nv[q] = src[ypos(j + q * TPR, N, mirror)];
        }
        F::run(v, c);
        if (cur_live) {
#pragma unroll
            for (int q = 0; q < R / 2; ++q) dst[q * TPR] = v[q];
        }
    }
}

// ------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------
// Per kernel instantiation: one PerDevice cache (hfft_internal.h) of the shared-memory opt-in and of the CTAs per SM
// the runtime reports for (threads, smem), keyed by device.
// persistent grid: `items` units of work in contiguous chunks of `per_cta`
static void chunk_grid(long long items, int num_sms, int occ, unsigned& grid, int& per_cta) {
    long long g = (long long)num_sms * occ;
    if (g > items) g = items;
    if (g < 1) g = 1;
    long long pc = (items + g - 1) / g;
    grid = (unsigned)((items + pc - 1) / pc);
    per_cta = (int)pc;
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

static int fft_tpr(int log2N) { return (1 << log2N) / (log2N < 3 ? (1 << log2N) : 8); }

// rows per block of the x kernels: a 128-byte run of the transposed X^, at most XCfg::MAXT threads
template <typename T> static int x_log2_rows_per_block(int log2N, int rows_per_plane) {
    const int tpr = fft_tpr(log2N);
    int rb = (int)(128 / sizeof(HFFT_C));
    while (rb > 1 && rb * tpr > XCfg<T>::MAXT) rb /= 2;
    while (rb > rows_per_plane) rb /= 2;
    int l = 0;
    while ((1 << l) < rb) ++l;
    return l;
}

template <typename T, bool ZP>
cudaError_t launch_fftx_fwd(const T* in, void* xhat, int log2nx, int nplanes, int rows_per_plane, int nz,
                            const double* ms_host, const void* tw, const void* twt, int num_sms, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2nx;
    const int log2rb = x_log2_rows_per_block<T>(log2nx, rows_per_plane), rb = 1 << log2rb;
    const int threads = rb * fft_tpr(log2nx);
    const size_t row_bytes = (size_t)2 * N * sizeof(C);
    const size_t smem = (rb + 1) * row_bytes;
    const long long nblocks = (long long)nplanes * rows_per_plane / rb;
    MsParam<T> ms;
    const int use_ms = ms_host != nullptr;
    for (int k = 0; k < HFFT_MAX_NZ; ++k) ms.v[k] = (use_ms && k < nz) ? (T)ms_host[k] : (T)1;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_X(log2nx, {
        auto kern = fftx_fwd_kernel<T, L, ZP>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int bpc;
            chunk_grid(nblocks, num_sms, occ, grid, bpc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, in, (C*)xhat, log2rb, rows_per_plane, nz > 0 ? nz : 1, use_ms, ms,
                                              (const C*)tw, (const C*)twt, nblocks, bpc);
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_ifftx(const void* xhat, T* out, int log2nx, int nplanes, int rows_per_plane, const void* tw,
                         const void* twt, int num_sms, const T* m, double* sums, cudaStream_t st) {
    typedef HFFT_C C;
    const int N = 1 << log2nx;
    const int log2rb = x_log2_rows_per_block<T>(log2nx, rows_per_plane), rb = 1 << log2rb;
    const int threads = rb * fft_tpr(log2nx);
    const size_t row_bytes = (size_t)2 * N * sizeof(C);
    const size_t smem = (rb + 1) * row_bytes + (size_t)(N + 1) * rb * sizeof(C);   // rows + alignment slack + X^ tile
    const long long nblocks = (long long)nplanes * rows_per_plane / rb;
    cudaError_t err = cudaErrorInvalidValue;
    if (sums) {
        HFFT_DISPATCH_X(log2nx, {
            auto kern = ifftx_kernel<T, L, true>;
            static PerDevice<int> lc;
            int occ = 1;
            if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
                unsigned grid; int bpc;
                chunk_grid(nblocks, num_sms, occ, grid, bpc);
                err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)xhat, out, log2rb, rows_per_plane, (const C*)tw,
                                                  (const C*)twt, nblocks, bpc, m, sums);
            }
        })
        return err;
    }
    HFFT_DISPATCH_X(log2nx, {
        auto kern = ifftx_kernel<T, L, false>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int bpc;
            chunk_grid(nblocks, num_sms, occ, grid, bpc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)xhat, out, log2rb, rows_per_plane, (const C*)tw,
                                              (const C*)twt, nblocks, bpc, m, sums);
        }
    })
    return err;
}

template <typename T, bool ZP>
cudaError_t launch_ffty_fwd(const void* xhat, void* spec, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                            const void* twt, int num_sms, cudaStream_t st, int mirror) {
    typedef HFFT_C C;
    const int N = 1 << log2N;
    const int tpr = fft_tpr(log2N);
    const int threads = tpr > 128 ? tpr : 128;
    const int rpc = threads / tpr;
    const long long nrows = (long long)nplanes * (nx + 1);
    const size_t row_bytes = (size_t)2 * N * sizeof(C);
    const size_t smem = (rpc + 1) * row_bytes;
    const long long ngroups = (nrows + rpc - 1) / rpc;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_Y(log2N, {
        auto kern = ffty_fwd_kernel<T, L, ZP>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int gpc;
            chunk_grid(ngroups, num_sms, occ, grid, gpc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)xhat, (C*)spec, nrows, nx + 1, nz_rot, ks, (const C*)twt,
                                              ngroups, gpc, mirror);
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_iffty(const void* spec, void* xhat, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                         const void* twt, int num_sms, cudaStream_t st, int mirror) {
    typedef HFFT_C C;
    const int N = 1 << log2N;
    const int tpr = fft_tpr(log2N);
    const int threads = tpr > 128 ? tpr : 128;
    const int rpc = threads / tpr;
    const long long nrows = (long long)nplanes * (nx + 1);
    const size_t row_bytes = (size_t)2 * N * sizeof(C);
    const size_t smem = (rpc + 1) * row_bytes;
    const long long ngroups = (nrows + rpc - 1) / rpc;
    cudaError_t err = cudaErrorInvalidValue;
    HFFT_DISPATCH_Y(log2N, {
        auto kern = iffty_kernel<T, L>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int gpc;
            chunk_grid(ngroups, num_sms, occ, grid, gpc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)spec, (C*)xhat, nrows, nx + 1, nz_rot, ks, (const C*)twt,
                                              ngroups, gpc, mirror);
        }
    })
    return err;
}

// explicit instantiations used by hfft_api.cu / tensor_build.cu
template cudaError_t launch_fftx_fwd<float, true>(const float*, void*, int, int, int, int, const double*, const void*, const void*, int, cudaStream_t);
template cudaError_t launch_fftx_fwd<double, true>(const double*, void*, int, int, int, int, const double*, const void*, const void*, int, cudaStream_t);
template cudaError_t launch_fftx_fwd<double, false>(const double*, void*, int, int, int, int, const double*, const void*, const void*, int, cudaStream_t);
template cudaError_t launch_ifftx<float>(const void*, float*, int, int, int, const void*, const void*, int, const float*, double*, cudaStream_t);
template cudaError_t launch_ifftx<double>(const void*, double*, int, int, int, const void*, const void*, int, const double*, double*, cudaStream_t);
template cudaError_t launch_ffty_fwd<float, true>(const void*, void*, int, int, int, int, long long, const void*, int, cudaStream_t, int);
template cudaError_t launch_ffty_fwd<double, true>(const void*, void*, int, int, int, int, long long, const void*, int, cudaStream_t, int);
template cudaError_t launch_ffty_fwd<double, false>(const void*, void*, int, int, int, int, long long, const void*, int, cudaStream_t, int);
template cudaError_t launch_iffty<float>(const void*, void*, int, int, int, int, long long, const void*, int, cudaStream_t, int);
template cudaError_t launch_iffty<double>(const void*, void*, int, int, int, int, long long, const void*, int, cudaStream_t, int);

}  // namespace hfft
