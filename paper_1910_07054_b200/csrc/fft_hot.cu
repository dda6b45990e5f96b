// fft_hot.cu -- the four FFT kernels of the hot path (stages S1, S2, S4, S5 of DESIGN.md), second generation.
//
//   S1 hfftx_fwd : M = Ms_j m (Eq.17); real-to-complex DFT of length 2nx of a row that is zero beyond nx
//                  (F_1 of Eq.23), kept for kx = 0..nx
//   S2 hffty_fwd : complex DFT of length 2ny along y (F_2 of Eq.24), rows >= ny zero
//   S4 hiffty    : inverse along y, only the first ny outputs (crop fused)
//   S5 hifftx    : complex-to-real inverse of length 2nx, only the first nx outputs
//
// Every transform is zero-padded or cropped, so it is done as TWO full transforms of HALF the length (subfft.cuh): the
// even and the odd outputs (forward) / the even and the odd cropped samples (inverse).  16 elements per thread in fp32
// (8 in fp64), radix 16 x 16: a 512-point padded transform is two 256-point ones with a single shared-memory exchange
// each, synchronised inside one warp.
//
// Layouts (C = complex of T):
//   real field  [plane][ny][nx]                 plane = (state, component, layer)
//   X^          [plane][ny][nx] C, kx fastest:  X^[kx], kx = 1..nx-1, and X^[0] = (DC, Nyquist) -- both are real, the
//               Nyquist term kx = nx rides in the imaginary part of kx = 0.  NOT transposed: the x kernels read and write
//               whole rows straight from / to registers (no staging, no CTA barrier); the y kernels take the strided side,
//               a tile of C = 8 columns x ny rows (64-byte runs) staged through shared memory -- asynchronously one tile
//               ahead on the way in (cp.async), one tile behind on the way out.
//   M^ / H^     [plane][KS] C, element kx * 2ny + ky, or the mirror layout kx * (2ny + 2) + ypos(ky) (fft.cuh: ypos);
//               kx = 0..nx.  The z planes hold i M_z / i H_z (real form R6) unless nz_rot == 0.
//
// x transforms (real data): the row of 2nx reals (nx non-zero) is packed as N = nx complex z[t] = x[2t] + i x[2t+1]
// (M = nx / 2 non-zero); Z = DFT_N(z) by the two half transforms; X[k] = E[k] + W_2N^k O[k] with
// E = (Z[k] + conj Z[N-k]) / 2, O = (Z[k] - conj Z[N-k]) / (2i).  k and N - k have the same parity, so the partner value
// sits in the same sub-transform, at lane TPR - j (even) / TPR - 1 - j (odd), register R - 1 - q: one warp shuffle.
// The inverse reads X[k], X[k + M], X[N - k], X[M - k] from the row (L1) and forms the sub-transform inputs directly.
#include "hfft_internal.h"
#include "subfft.cuh"

namespace hfft {

#ifndef HFFT_YC_TPR
#define HFFT_YC_TPR 64
#endif
template <typename T> struct HotCfg {
    static constexpr int LOG2RMAX = sizeof(T) == 4 ? 4 : 3;
    static constexpr bool REGTW = sizeof(T) == 4;
};

__device__ __forceinline__ unsigned hot_smem_base(unsigned align) {
    extern __shared__ __align__(16) unsigned char hot_smem_raw[];
    return (smem_u32(hot_smem_raw) + align - 1) & ~(align - 1);
}

__device__ __forceinline__ float2 shfl_c(float2 v, int src) {
    float2 r;
    r.x = __shfl_sync(0xffffffffu, v.x, src);
    r.y = __shfl_sync(0xffffffffu, v.y, src);
    return r;
}
__device__ __forceinline__ double2 shfl_c(double2 v, int src) {
    double2 r;
    r.x = __shfl_sync(0xffffffffu, v.x, src);
    r.y = __shfl_sync(0xffffffffu, v.y, src);
    return r;
}

__device__ __forceinline__ void cp_async_elem(unsigned dst, const float2* src) {
    asm volatile("cp.async.ca.shared.global.L2::128B [%0], [%1], 8;\n" ::"r"(dst), "l"(src));
}
__device__ __forceinline__ void cp_async_elem(unsigned dst, const double2* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(src));
}

// ------------------------------------------------------------------------------------------
// S1: forward x.  Thread (row slot r, half h, j); one pass handles blockDim / (2 TPR) rows.
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2M>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? 2 : 1)
hfftx_fwd_kernel(const T* __restrict__ in, HFFT_C* __restrict__ xhat, int rows_per_plane, int nz, int use_ms,
                 MsParam<T> ms, const HFFT_C* __restrict__ tw /* exp(-2 pi i t / 2N), 2N entries, N = 2M */,
                 const HFFT_C* __restrict__ twt, long long nrows, int rpc) {
    typedef HFFT_C C;
    typedef SubFFT<T, LOG2M, false, HotCfg<T>::LOG2RMAX, HotCfg<T>::REGTW> F;
    constexpr int M = F::M, R = F::R, TPR = F::TPR, N = 2 * M;
    constexpr int CQ = 32 / R;                                // exp(-2 pi i q / (2R)) = 64th root number q * CQ
    const int tid = threadIdx.x, lane = tid & 31;
    const int j = tid & (TPR - 1), h = (tid >> F::LOG2TPR) & 1, r = tid >> (F::LOG2TPR + 1);
    const int rb = blockDim.x >> (F::LOG2TPR + 1);
    typename F::Ctx c;
    F::init(c, hot_smem_base(F::SUB_BYTES) + (unsigned)(2 * r + h) * F::SUB_BYTES, j, twt);
    const C wpre = __ldg(tw + 2 * j);                          // w_N^j
    const C wsplit = __ldg(tw + 2 * j + h);                    // W_2N^(2j + h)
    const int plane_lane = (lane & ~(TPR - 1) & 31) | ((h ? (TPR - 1 - j) : ((TPR - j) & (TPR - 1))) & 31);
    const bool self0 = h == 0 && j == 0;

    const long long row0 = (long long)blockIdx.x * rpc;
    const long long rend = row0 + rpc < nrows ? row0 + rpc : nrows;
    const int nit = (int)((rend - row0 + rb - 1) / rb);
    pdl_wait();                                               // the previous kernel of the stream may still write `in`
    for (int it = 0; it < nit; ++it) {
        const long long row = row0 + (long long)it * rb + r;
        const bool live = row < rend;
        const C* zin = reinterpret_cast<const C*>(in) + row * M + j;
        C v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = live ? zin[q * TPR] : mk<T>(0, 0);
        if (use_ms) {
            const T sc = ms.v[live ? (int)((row / rows_per_plane) % nz) : 0];
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = cscale(sc, v[q]);
        }
        if (h) {                                              // odd outputs: x[n] w_N^n, n = j + q TPR
            static_for<0, R>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                v[q] = mul_root64<q * CQ, false>(cmul(v[q], wpre));
            });
        }
        F::run(v, c);                                         // v[q] = Z[2 (j + q TPR) + h]
        if constexpr (TPR > 32) {                             // the partner lives in another warp: through the buffer
#pragma unroll
            for (int q = 0; q < R; ++q) sts(c.ld ^ ((unsigned)F::swz(q * TPR) << F::SH), v[q]);
            __syncthreads();
        }
        C* xrow = xhat + row * N + 2 * j + h;
        static_for<0, R>([&](auto qc) {
            constexpr int q = decltype(qc)::value;
            C o;
            if constexpr (TPR > 32) {                         // Z[2 m' + h], m' = M - m - h (mod M), m = j + q TPR
                const int pm = (M - h - (j + q * TPR)) & (M - 1);
                o = lds<C>(c.ld ^ ((unsigned)(F::swz(j) ^ F::swz(pm)) << F::SH));
            } else {
                o = shfl_c(v[R - 1 - q], plane_lane);
                if (self0) o = v[(R - q) % R];
            }
            const C zk = v[q], zn = cconj(o);
            const C s = cadd(zk, zn);                                                      // 2 E
            const C wo = mul_root64<q * CQ, false>(cmul(mul_mi(csub(zk, zn)), wsplit));    // 2 W O
            C x = cscale((T)0.5, cadd(s, wo));
            if (q == 0 && self0) x = mk<T>(zk.x + zk.y, zk.x - zk.y);                      // (DC, Nyquist)
            if (live) xrow[2 * q * TPR] = x;
        });
        if constexpr (TPR > 32) __syncthreads();              // the buffer is read before the next row's exchange
    }
}

// ------------------------------------------------------------------------------------------
// S5: inverse x (complex-to-real, crop to the first nx reals = first M complex outputs).
// Z~[k] = E~ + i O~,  E~ = X[k] + conj X[N-k],  O~ = (X[k] - conj X[N-k]) W_2N^{-k};  z~ = IDFT_N(Z~) cropped.
// RED (hfft_plan_set_reduction): also accumulates, per plane, the sum of h and of m h (doubles).
// ------------------------------------------------------------------------------------------
template <typename T, int LOG2M, bool RED>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? 2 : 1)
hifftx_kernel(const HFFT_C* __restrict__ xhat, T* __restrict__ out, int rows_per_plane, const HFFT_C* __restrict__ tw,
              const HFFT_C* __restrict__ twt, long long nrows, int rpc, const T* __restrict__ m, double* __restrict__ sums) {
    typedef HFFT_C C;
    typedef SubFFT<T, LOG2M, true, HotCfg<T>::LOG2RMAX, HotCfg<T>::REGTW> F;
    constexpr int M = F::M, R = F::R, TPR = F::TPR, N = 2 * M;
    constexpr int RS = R > 1 ? R / 2 : 1;                     // stored outputs per thread (crop)
    const int tid = threadIdx.x;
    const int j = tid & (TPR - 1), h = (tid >> F::LOG2TPR) & 1, r = tid >> (F::LOG2TPR + 1);
    const int rb = blockDim.x >> (F::LOG2TPR + 1);
    typename F::Ctx c;
    F::init(c, hot_smem_base(F::SUB_BYTES) + (unsigned)(2 * r + h) * F::SUB_BYTES, j, twt);
    const C wj = __ldg(tw + j);                                // W_2N^j
    const C w2j = __ldg(tw + 2 * j);                           // w_N^j

    const long long row0 = (long long)blockIdx.x * rpc;
    const long long rend = row0 + rpc < nrows ? row0 + rpc : nrows;
    const int nit = (int)((rend - row0 + rb - 1) / rb);
    pdl_wait();                                               // X^ comes from the previous kernel (S4)
    for (int it = 0; it < nit; ++it) {
        const long long row = row0 + (long long)it * rb + r;
        const bool live = row < rend;
        const C* X = xhat + (live ? row : row0) * N;
        C v[R];
        static_for<0, R>([&](auto qc) {
            constexpr int q = decltype(qc)::value;
            const int k = j + q * TPR;
            C P = X[k], Pp = X[k + M], Q = cconj(X[(N - k) & (N - 1)]), Qp = cconj(X[M - k]);
            if (q == 0 && j == 0) { Q = mk<T>(P.y, 0); P = mk<T>(P.x, 0); }                // DC and Nyquist (both real)
            // conj(W_2N^k) through cmulc; W_2N^k = W_2N^j exp(-2 pi i q / (4R))
            const C zk = cadd(cadd(P, Q), mul_pi(mul_root64<q * (16 / R), true>(cmulc(csub(P, Q), wj))));
            const C zm = csub(cadd(Pp, Qp), mul_root64<q * (16 / R), true>(cmulc(csub(Pp, Qp), wj)));
            v[q] = h ? mul_root64<q * (32 / R), true>(cmulc(csub(zk, zm), w2j)) : cadd(zk, zm);
        });
        F::run(v, c);                                         // v[q] = z[2 (j + q TPR) + h]
        C* zout = reinterpret_cast<C*>(out) + row * M + 2 * j + h;
        const bool st = live && (R > 1 || h == 0);
        if (st) {
#pragma unroll
            for (int q = 0; q < RS; ++q) zout[2 * q * TPR] = v[q];
        }
        if constexpr (RED) {
            double sh = 0.0, smh = 0.0;
            if (st) {
                const C* zm = reinterpret_cast<const C*>(m) + row * M + 2 * j + h;
#pragma unroll
                for (int q = 0; q < RS; ++q) {
                    const C mm = zm[2 * q * TPR];
                    sh += (double)v[q].x + (double)v[q].y;
                    smh += (double)v[q].x * (double)mm.x + (double)v[q].y * (double)mm.y;
                }
            }
            // the lanes of a warp may belong to rows of different planes: reduce over the row's own 2 TPR lanes only
            constexpr int GRP = 2 * TPR < 32 ? 2 * TPR : 32;
#pragma unroll
            for (int o = GRP / 2; o > 0; o >>= 1) {
                sh += __shfl_xor_sync(0xffffffffu, sh, o);
                smh += __shfl_xor_sync(0xffffffffu, smh, o);
            }
            if (live && (tid & (GRP - 1)) == 0) {
                const long long plane = row / rows_per_plane;
                atomicAdd(sums + 2 * plane, sh);
                atomicAdd(sums + 2 * plane + 1, smh);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// S2 / S4: transforms along y.  A tile = NC = 8 columns (kx0 .. kx0 + 7) of one plane, all ny rows.  Thread (column slot
// cc, half h, j).  Staging tile [ny][NC] in shared memory; element (y, c) lives at row y ^ ((y >> 4) & 1), slot
// c ^ ((y >> 1) & 7): conflict free for the copy side (lanes along c, then y), for the column reads of S2 (16
// consecutive y) and for the column writes of S4 (16 y of one parity).  Every index is (per-thread part) | (compile-time
// part) on disjoint bits and the placement is XOR-linear in the low bits, additive in the high ones, so an address is
// ((per-thread base) XOR constant) + constant: one LOP3 per shared-memory access, like the exchanges of subfft.cuh.
// ------------------------------------------------------------------------------------------
template <int LOG2C> struct TileMap {
    static constexpr int NC = 1 << LOG2C;
    // element index inside the tile = hi(y) + lo(y, c); a pair of rows holds 2 NC elements
    static __host__ __device__ constexpr int lo(int y, int c) { return (((y ^ (y >> 4)) & 1) << LOG2C) | ((c ^ (y >> 1)) & (NC - 1)); }
    static __host__ __device__ constexpr int hi(int y) { return (y >> 1) * 2 * NC; }
};

// CTA shape of the y kernels: NC columns x 2 halves x TPR threads; 8 columns, fewer where that would exceed 512 threads
// (the register budget of 16 complex values per thread)
template <typename T, int LOG2M> struct YHot {
    static constexpr int TPR = SubFFT<T, LOG2M, false, HotCfg<T>::LOG2RMAX, true>::TPR;
    static constexpr int LOG2C = TPR >= 128 ? 1 : (TPR >= HFFT_YC_TPR ? 2 : 3);
    static constexpr int THREADS = (2 * TPR) << LOG2C;
    static constexpr int MAXT = THREADS < 256 ? 256 : THREADS;
};

template <typename T, int LOG2M>
__global__ void __launch_bounds__(YHot<T, LOG2M>::MAXT)
hffty_fwd_kernel(const HFFT_C* __restrict__ xhat, HFFT_C* __restrict__ spec, long long nplanes, int nx, int log2tx,
                 int nz_rot, long long ks, const HFFT_C* __restrict__ twy /* exp(-2 pi i t / 2M), 2M entries */,
                 const HFFT_C* __restrict__ twt, long long ntiles, int tpc, int mirror) {
    typedef HFFT_C C;
    typedef SubFFT<T, LOG2M, false, HotCfg<T>::LOG2RMAX, HotCfg<T>::REGTW> F;
    typedef TileMap<YHot<T, LOG2M>::LOG2C> TM;
    constexpr int M = F::M, R = F::R, TPR = F::TPR, LOG2C = YHot<T, LOG2M>::LOG2C, NC = 1 << LOG2C;
    constexpr int CQ = 32 / R;
    constexpr int ES = (int)sizeof(C);
    constexpr int YSTEP = 2 * TPR, NI = M / YSTEP;            // copy side: thread (y0 = tid / NC, cx), rows y0 + i YSTEP
    constexpr unsigned STG_BYTES = (unsigned)(M << LOG2C) * ES;
    const int tid = threadIdx.x;
    const int j = tid & (TPR - 1), h = (tid >> F::LOG2TPR) & 1, cc = tid >> (F::LOG2TPR + 1);
    const int cx = tid & (NC - 1), y0 = tid >> LOG2C;
    const unsigned base = hot_smem_base(F::SUB_BYTES > 2 * NC * ES ? F::SUB_BYTES : 2 * NC * ES);
    typename F::Ctx c;
    F::init(c, base + (unsigned)(2 * cc + h) * F::SUB_BYTES, j, twt);
    const unsigned stg = base + (unsigned)(2 * NC) * F::SUB_BYTES;
    const unsigned rd0 = stg + (unsigned)(TM::hi(j) + TM::lo(j, cc)) * ES;       // column read: element (j + q TPR, cc)
    const unsigned cp0 = stg + (unsigned)(TM::hi(y0) + TM::lo(y0, cx)) * ES;     // copy: element (y0 + i YSTEP, cx)
    const C wpre = __ldg(twy + j);                             // w_2M^j
    const long long regular = nplanes << log2tx;
    const int pitch = mirror ? 2 * M + 2 : 2 * M;
    // spectrum slots of ky = 2 (j + q TPR) + h: plain ky; mirror 2 ky for ky <= M, else 2 (2M - ky) + 1
    const int offa = mirror ? 4 * j + 2 * h : 2 * j + h;
    const int offb = mirror ? 4 * M + 1 - 4 * j - 2 * h : 2 * j + h;
    const int stra = mirror ? 4 * TPR : 2 * TPR, strb = mirror ? -4 * TPR : 2 * TPR;

    const long long t0 = (long long)blockIdx.x * tpc;
    const int nit = (int)((ntiles - t0 < tpc) ? ntiles - t0 : tpc);
    auto fetch = [&](long long t, int buf) {
        const unsigned dst = cp0 + buf * STG_BYTES;
        if (t < regular) {
            const long long plane = t >> log2tx;
            const int kx = ((int)(t - (plane << log2tx)) << LOG2C) + cx;
            const C* src = xhat + (plane * M + y0) * nx + kx;
            if (kx < nx) {
                static_for<0, NI>([&](auto ic) {
                    constexpr int yb = decltype(ic)::value * YSTEP;
                    cp_async_elem((dst ^ (unsigned)(TM::lo(yb, 0) * ES)) + (unsigned)(TM::hi(yb) * ES), src + (long long)yb * nx);
                });
            }
        } else {                                              // Nyquist columns of planes pl0 + cx: Im X^[.][y][0]
            const long long pl = ((t - regular) << LOG2C) + cx;
            static_for<0, NI>([&](auto ic) {
                constexpr int yb = decltype(ic)::value * YSTEP;
                const T vy = pl < nplanes ? xhat[(pl * M + y0 + yb) * nx].y : (T)0;
                sts((dst ^ (unsigned)(TM::lo(yb, 0) * ES)) + (unsigned)(TM::hi(yb) * ES), mk<T>(vy, 0));
            });
        }
        cp_async_commit();
    };
    pdl_wait();                                               // X^ comes from the previous kernel (S1)
    if (nit > 0) fetch(t0, 0);
    for (int it = 0; it < nit; ++it) {
        cp_async_wait_group<0>();
        __syncthreads();                                      // tile `it` has landed; everyone is done with tile it - 1
        if (it + 1 < nit) fetch(t0 + it + 1, (it + 1) & 1);
        const long long t = t0 + it;
        const bool extra = t >= regular;
        const long long plane = extra ? ((t - regular) << LOG2C) + cc : (t >> log2tx);
        const int kx = extra ? nx : ((int)(t - (plane << log2tx)) << LOG2C) + cc;
        const bool live = plane < nplanes && kx <= nx && (extra || kx < nx);
        const unsigned src = rd0 + (it & 1) * STG_BYTES;
        C v[R];
        static_for<0, R>([&](auto qc) {
            constexpr int yb = decltype(qc)::value * TPR;
            v[decltype(qc)::value] = lds<C>((src ^ (unsigned)(TM::lo(yb, 0) * ES)) + (unsigned)(TM::hi(yb) * ES));
        });
        if (kx == 0) {                                        // X^[0] = (DC, Nyquist): this column is the DC term
#pragma unroll
            for (int q = 0; q < R; ++q) v[q].y = 0;
        }
        if (h) {
            static_for<0, R>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                v[q] = mul_root64<q * CQ, false>(cmul(v[q], wpre));
            });
        }
        F::run(v, c);                                         // v[q] = Y[2 (j + q TPR) + h]
        if (live) {
            if (nz_rot > 0 && (int)(plane % (3 * nz_rot)) >= 2 * nz_rot) {     // M'_z = i M_z
#pragma unroll
                for (int q = 0; q < R; ++q) v[q] = mul_pi(v[q]);
            }
            C* dst = spec + plane * ks + (long long)kx * pitch;
            // q < R / 2: ky < M.  q >= R / 2: ky >= M, and ky == M only for j = 0, h = 0, q = R / 2
            static_for<0, R>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                if constexpr (2 * q < R) dst[offa + q * stra] = v[q];
                else if constexpr (2 * q == R) dst[(j | h) == 0 ? (mirror ? 2 * M : M) : offb + q * strb] = v[q];
                else dst[offb + q * strb] = v[q];
            });
        }
    }
}

template <typename T, int LOG2M>
__global__ void __launch_bounds__(YHot<T, LOG2M>::MAXT)
hiffty_kernel(const HFFT_C* __restrict__ spec, HFFT_C* __restrict__ xhat, long long nplanes, int nx, int log2tx,
              int nz_rot, long long ks, const HFFT_C* __restrict__ twy, const HFFT_C* __restrict__ twt,
              long long ntiles, int tpc, int mirror) {
    typedef HFFT_C C;
    typedef SubFFT<T, LOG2M, true, HotCfg<T>::LOG2RMAX, HotCfg<T>::REGTW> F;
    typedef TileMap<YHot<T, LOG2M>::LOG2C> TM;
    constexpr int M = F::M, R = F::R, TPR = F::TPR, LOG2C = YHot<T, LOG2M>::LOG2C, NC = 1 << LOG2C;
    constexpr int CQ = 32 / R;
    constexpr int RS = R / 2;                                 // kept outputs per thread (M >= 2, so R >= 2)
    constexpr int ES = (int)sizeof(C);
    constexpr int YSTEP = 2 * TPR, NI = M / YSTEP;
    constexpr unsigned STG_BYTES = (unsigned)(M << LOG2C) * ES;
    const int tid = threadIdx.x;
    const int j = tid & (TPR - 1), h = (tid >> F::LOG2TPR) & 1, cc = tid >> (F::LOG2TPR + 1);
    const int cx = tid & (NC - 1), y0 = tid >> LOG2C;
    const unsigned base = hot_smem_base(F::SUB_BYTES > 2 * NC * ES ? F::SUB_BYTES : 2 * NC * ES);
    typename F::Ctx c;
    F::init(c, base + (unsigned)(2 * cc + h) * F::SUB_BYTES, j, twt);
    const unsigned stg = base + (unsigned)(2 * NC) * F::SUB_BYTES;
    const unsigned wr0 = stg + (unsigned)(TM::hi(2 * j + h) + TM::lo(2 * j + h, cc)) * ES;   // element (2 (j + q TPR) + h, cc)
    const unsigned cp0 = stg + (unsigned)(TM::hi(y0) + TM::lo(y0, cx)) * ES;
    const C wj = __ldg(twy + j);                               // w_2M^j
    const int pitch = mirror ? 2 * M + 2 : 2 * M;
    // spectrum slots of k = j + q TPR (< M) and of k + M; k + M == M only for k = 0
    const int offa = mirror ? 2 * j : j, stra = mirror ? 2 * TPR : TPR;
    const int offb = mirror ? 2 * M + 1 - 2 * j : M + j, strb = mirror ? -2 * TPR : TPR;

    const long long t0 = (long long)blockIdx.x * tpc;
    const int nit = (int)((ntiles - t0 < tpc) ? ntiles - t0 : tpc);
    pdl_wait();                                               // H^ comes from the previous kernel (S3)
    for (int it = 0; it < nit; ++it) {
        const long long t = t0 + it;
        const long long plane = t >> log2tx;
        const int kx0 = (int)(t - (plane << log2tx)) << LOG2C, kx = kx0 + cc;
        const bool live = kx < nx;
        const C* src = spec + plane * ks + (long long)(live ? kx : 0) * pitch;
        const C* srcn = spec + plane * ks + (long long)nx * pitch;             // kx = nx: joins kx = 0 as its imaginary part
        const bool rot = nz_rot > 0 && (int)(plane % (3 * nz_rot)) >= 2 * nz_rot;
        C v[R];
        static_for<0, R>([&](auto qc) {
            constexpr int q = decltype(qc)::value;
            const int pa = offa + q * stra;
            const int pb = (q == 0 && j == 0) ? (mirror ? 2 * M : M) : offb + q * strb;
            C A = src[pa], B = src[pb];
            if (kx == 0) { A = cadd(A, mul_pi(srcn[pa])); B = cadd(B, mul_pi(srcn[pb])); }
            if (rot) { A = mul_mi(A); B = mul_mi(B); }                         // H_z = -i H'_z
            v[q] = h ? mul_root64<q * CQ, true>(cmulc(csub(A, B), wj)) : cadd(A, B);
        });
        F::run(v, c);                                         // v[q] = z[2 (j + q TPR) + h], q < R / 2 kept
        const unsigned dst = wr0 + (it & 1) * STG_BYTES;
        static_for<0, RS>([&](auto qc) {
            constexpr int yb = 2 * decltype(qc)::value * TPR;
            sts((dst ^ (unsigned)(TM::lo(yb, 0) * ES)) + (unsigned)(TM::hi(yb) * ES), v[decltype(qc)::value]);
        });
        __syncthreads();                                      // tile complete; the other buffer's copy-out is over too
        if (kx0 + cx < nx) {
            C* out = xhat + (plane * M + y0) * nx + kx0 + cx;
            const unsigned rd = cp0 + (it & 1) * STG_BYTES;
            static_for<0, NI>([&](auto ic) {
                constexpr int yb = decltype(ic)::value * YSTEP;
                out[(long long)yb * nx] = lds<C>((rd ^ (unsigned)(TM::lo(yb, 0) * ES)) + (unsigned)(TM::hi(yb) * ES));
            });
        }
    }
}

// ------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------
static void hot_chunk_grid(long long items, int num_sms, int occ, unsigned& grid, int& per_cta) {
    long long g = (long long)num_sms * occ;
    if (g > items) g = items;
    if (g < 1) g = 1;
    const long long pc = (items + g - 1) / g;
    grid = (unsigned)((items + pc - 1) / pc);
    per_cta = (int)pc;
}

#define HOT_CASE(V, ...) case V: { constexpr int L = V; __VA_ARGS__ } break;
#define HOT_DISPATCH(LG, ...)                                                                                     \
    switch (LG) {                                                                                                 \
        HOT_CASE(0, __VA_ARGS__) HOT_CASE(1, __VA_ARGS__) HOT_CASE(2, __VA_ARGS__) HOT_CASE(3, __VA_ARGS__)       \
        HOT_CASE(4, __VA_ARGS__) HOT_CASE(5, __VA_ARGS__) HOT_CASE(6, __VA_ARGS__) HOT_CASE(7, __VA_ARGS__)       \
        HOT_CASE(8, __VA_ARGS__) HOT_CASE(9, __VA_ARGS__)                                                         \
        default: break;                                                                                           \
    }
#define HOT_DISPATCH_Y(LG, ...)                                                                                   \
    switch (LG) {                                                                                                 \
        HOT_CASE(1, __VA_ARGS__) HOT_CASE(2, __VA_ARGS__) HOT_CASE(3, __VA_ARGS__) HOT_CASE(4, __VA_ARGS__)       \
        HOT_CASE(5, __VA_ARGS__) HOT_CASE(6, __VA_ARGS__) HOT_CASE(7, __VA_ARGS__) HOT_CASE(8, __VA_ARGS__)       \
        HOT_CASE(9, __VA_ARGS__) HOT_CASE(10, __VA_ARGS__)                                                        \
        default: break;                                                                                           \
    }

template <typename T> static int hot_tpr(int log2m) {
    const int lr = log2m < HotCfg<T>::LOG2RMAX ? log2m : HotCfg<T>::LOG2RMAX;
    return 1 << (log2m - lr);
}

// x kernels: rows per pass so that a CTA has 256 threads (fewer when there are not that many rows)
template <typename T> static void hot_x_shape(int log2m, long long nrows, int& threads, size_t& smem) {
    const int tpr = hot_tpr<T>(log2m);
    int rb = 256 / (2 * tpr);
    if (rb < 1) rb = 1;
    while (rb > 1 && rb > nrows) rb /= 2;
    threads = rb * 2 * tpr;
    const size_t sub = ((size_t)1 << log2m) * 2 * sizeof(T);
    smem = (size_t)(2 * rb + 1) * sub;
}

template <typename T>
cudaError_t launch_hfftx_fwd(const T* in, void* xhat, int log2nx, int nplanes, int rows_per_plane, int nz,
                             const double* ms_host, const void* tw, const void* twt, int num_sms, cudaStream_t st) {
    typedef HFFT_C C;
    const long long nrows = (long long)nplanes * rows_per_plane;
    int threads; size_t smem;
    hot_x_shape<T>(log2nx - 1, nrows, threads, smem);
    const int rb = threads / (2 * hot_tpr<T>(log2nx - 1));
    MsParam<T> ms;
    const int use_ms = ms_host != nullptr;
    for (int k = 0; k < HFFT_MAX_NZ; ++k) ms.v[k] = (use_ms && k < nz) ? (T)ms_host[k] : (T)1;
    cudaError_t err = cudaErrorInvalidValue;
    HOT_DISPATCH(log2nx - 1, {
        auto kern = hfftx_fwd_kernel<T, L>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int ppc;
            hot_chunk_grid((nrows + rb - 1) / rb, num_sms, occ, grid, ppc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, in, (C*)xhat, rows_per_plane, nz > 0 ? nz : 1, use_ms, ms,
                             (const C*)tw, (const C*)twt, nrows, ppc * rb);
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_hifftx(const void* xhat, T* out, int log2nx, int nplanes, int rows_per_plane, const void* tw,
                          const void* twt, int num_sms, const T* m, double* sums, cudaStream_t st) {
    typedef HFFT_C C;
    const long long nrows = (long long)nplanes * rows_per_plane;
    int threads; size_t smem;
    hot_x_shape<T>(log2nx - 1, nrows, threads, smem);
    const int rb = threads / (2 * hot_tpr<T>(log2nx - 1));
    cudaError_t err = cudaErrorInvalidValue;
    if (sums) {
        HOT_DISPATCH(log2nx - 1, {
            auto kern = hifftx_kernel<T, L, true>;
            static PerDevice<int> lc;
            int occ = 1;
            if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
                unsigned grid; int ppc;
                hot_chunk_grid((nrows + rb - 1) / rb, num_sms, occ, grid, ppc);
                err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)xhat, out, rows_per_plane, (const C*)tw,
                                 (const C*)twt, nrows, ppc * rb, m, sums);
            }
        })
        return err;
    }
    HOT_DISPATCH(log2nx - 1, {
        auto kern = hifftx_kernel<T, L, false>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int ppc;
            hot_chunk_grid((nrows + rb - 1) / rb, num_sms, occ, grid, ppc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)xhat, out, rows_per_plane, (const C*)tw,
                             (const C*)twt, nrows, ppc * rb, m, sums);
        }
    })
    return err;
}

// y kernels: tiles of NC columns (YHot); a CTA = NC columns x 2 halves x TPR threads.  nx < NC: one partly used tile per plane
template <typename T> static void hot_y_shape(int log2m, int nx, int& log2c, int& log2tx, int& threads, size_t& smem) {
    const int tpr = hot_tpr<T>(log2m);
    log2c = tpr >= 128 ? 1 : (tpr >= HFFT_YC_TPR ? 2 : 3);
    threads = (1 << log2c) * 2 * tpr;
    log2tx = 0;
    while (((1 << log2c) << log2tx) < nx) ++log2tx;
    const size_t es = 2 * sizeof(T);
    size_t sub = ((size_t)1 << log2m) * es;
    const size_t align = sub > 2 * ((size_t)1 << log2c) * es ? sub : 2 * ((size_t)1 << log2c) * es;
    smem = align + (size_t)(2 * (1 << log2c)) * sub + 2 * (((size_t)1 << log2m) << log2c) * es;
}

template <typename T>
cudaError_t launch_hffty_fwd(const void* xhat, void* spec, int nx, int log2ny, int nplanes, int nz_rot, long long ks,
                             const void* twy, const void* twt, int num_sms, cudaStream_t st, int mirror) {
    typedef HFFT_C C;
    int log2c, log2tx, threads; size_t smem;
    hot_y_shape<T>(log2ny, nx, log2c, log2tx, threads, smem);
    const long long ntiles = ((long long)nplanes << log2tx) + (((long long)nplanes + (1 << log2c) - 1) >> log2c);
    cudaError_t err = cudaErrorInvalidValue;
    HOT_DISPATCH_Y(log2ny, {
        auto kern = hffty_fwd_kernel<T, L>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int tpc;
            hot_chunk_grid(ntiles, num_sms, occ, grid, tpc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)xhat, (C*)spec, (long long)nplanes, nx, log2tx,
                             nz_rot, ks, (const C*)twy, (const C*)twt, ntiles, tpc, mirror);
        }
    })
    return err;
}

template <typename T>
cudaError_t launch_hiffty(const void* spec, void* xhat, int nx, int log2ny, int nplanes, int nz_rot, long long ks,
                          const void* twy, const void* twt, int num_sms, cudaStream_t st, int mirror) {
    typedef HFFT_C C;
    int log2c, log2tx, threads; size_t smem;
    hot_y_shape<T>(log2ny, nx, log2c, log2tx, threads, smem);
    const long long ntiles = (long long)nplanes << log2tx;
    cudaError_t err = cudaErrorInvalidValue;
    HOT_DISPATCH_Y(log2ny, {
        auto kern = hiffty_kernel<T, L>;
        static PerDevice<int> lc;
        int occ = 1;
        if ((err = ctas_per_sm_cached(kern, threads, smem, lc, occ)) == cudaSuccess) {
            unsigned grid; int tpc;
            hot_chunk_grid(ntiles, num_sms, occ, grid, tpc);
            err = launch_pdl(kern, dim3(grid), dim3(threads), smem, st, (const C*)spec, (C*)xhat, (long long)nplanes, nx, log2tx,
                             nz_rot, ks, (const C*)twy, (const C*)twt, ntiles, tpc, mirror);
        }
    })
    return err;
}

template cudaError_t launch_hfftx_fwd<float>(const float*, void*, int, int, int, int, const double*, const void*, const void*, int, cudaStream_t);
template cudaError_t launch_hfftx_fwd<double>(const double*, void*, int, int, int, int, const double*, const void*, const void*, int, cudaStream_t);
template cudaError_t launch_hifftx<float>(const void*, float*, int, int, int, const void*, const void*, int, const float*, double*, cudaStream_t);
template cudaError_t launch_hifftx<double>(const void*, double*, int, int, int, const void*, const void*, int, const double*, double*, cudaStream_t);
template cudaError_t launch_hffty_fwd<float>(const void*, void*, int, int, int, int, long long, const void*, const void*, int, cudaStream_t, int);
template cudaError_t launch_hffty_fwd<double>(const void*, void*, int, int, int, int, long long, const void*, const void*, int, cudaStream_t, int);
template cudaError_t launch_hiffty<float>(const void*, void*, int, int, int, int, long long, const void*, const void*, int, cudaStream_t, int);
template cudaError_t launch_hiffty<double>(const void*, void*, int, int, int, int, long long, const void*, const void*, int, cudaStream_t, int);

}  // namespace hfft
