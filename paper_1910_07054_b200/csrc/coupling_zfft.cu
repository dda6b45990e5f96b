// coupling_zfft.cu -- stage S3 for stacks of EQUAL layer thickness by the method the paper compares
// against: the z-convolution is also done by FFT, Eq.25
//
//     H = - F3^-1 [ F3(N) F3(M) ],
//
// here with the in-plane transforms already done by S1/S2 (and undone by S4/S5), so that S3 is, per
// in-plane wavevector k and component, a zero-padded FFT of length Lz >= 2 nz along z, a real
// symmetric 3 x 3 multiply per (k, kz), and the inverse FFT cropped to the nz layers:
// O(nz log nz) per wavevector instead of the O(nz^2) of the explicit sum.
//
// Bank (zdft_bank_kernel, setup): with g_d the in-plane spectra of the Toeplitz classes d = i - j
// (real a^c_d for xx, yy, zz, xy, even in d; i a^c_d for xz, yz, odd in d; the factor -1/(4 nx ny)
// folded, tensor_build.cu), on the periodic grid of length Lz (slot d = Lz/2 unused = 0):
//     S^c(kz) = [ a^c_0 + 2 sum_{d>0} a^c_d cos(2 pi kz d / Lz) ] / Lz      c = xx, yy, zz, xy
//     S^c(kz) = [         2 sum_{d>0} a^c_d sin(2 pi kz d / Lz) ] / Lz      c = xz, yz   (i * (-i) = 1)
// all real: H^(k, kz) = S(k, kz) M^(k, kz) with S the symmetric matrix [[xx,xy,xz],[xy,yy,yz],[xz,yz,zz]]
// acting on the UNROTATED spectra (S2 / S4 run with nz_rot = 0 in this mode).
// The cosine sums are even in kz and the sine sums odd, S^c(Lz - kz) = +- S^c(kz), so only kz = 0 .. Lz / 2 is stored:
// layout [tile][kz <= Lz/2][6][32] in the plan precision, 6 (Lz / 2 + 1) reals per wavevector, every value read once
// per evaluation (128 B per warp); kz > Lz / 2 uses slot Lz - kz with xz, yz negated.
//
// Kernel: lane = wavevector (global accesses are 256 B per warp along k), warp t of the TT warps of
// a CTA owns the layers n = t + TT q, q < E (Lz = E TT).  Forward (decimation in frequency):
//     Y[t][r] = W_Lz^{t r} sum_q x[t + TT q] W_E^{q r}          in registers (upper half of q is zero)
//     X[r + E s] = sum_t Y[t][r] W_TT^{t s}                     after ONE exchange through shared memory
// (thread t' takes r = t' E/TT ... and all t), multiply, and the same two steps backwards.
#include "hfft_internal.h"
#include "fft.cuh"

namespace hfft {

// DFT of N <= 16 points in registers, natural order in and out; ZH: v[N/2 ..] are zero on entry
template <int N, bool INV, bool ZH, typename T, typename C>
__device__ __forceinline__ void rdft(C* v) {
    if constexpr (N == 2) dft2<INV, ZH>(v[0], v[1]);
    else if constexpr (N == 4) dft4<INV, ZH>(v[0], v[1], v[2], v[3]);
    else if constexpr (N == 8) dft8<INV, ZH, T>(v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7]);
    else if constexpr (N == 16) {
        // X[2m] = DFT8(a_n + a_{n+8})[m], X[2m+1] = DFT8((a_n - a_{n+8}) W16^n)[m]
        const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173, h = (T)0.70710678118654752440;
        C e[8], o[8];
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            if (ZH) { e[n] = v[n]; o[n] = v[n]; }
            else { e[n] = cadd(v[n], v[n + 8]); o[n] = csub(v[n], v[n + 8]); }
        }
        o[1] = tmul<INV>(o[1], mk<T>(c1, -s1));
        o[2] = tmul<INV>(o[2], mk<T>(h, -h));
        o[3] = tmul<INV>(o[3], mk<T>(s1, -c1));
        o[4] = mul_qt<INV>(o[4]);
        o[5] = tmul<INV>(o[5], mk<T>(-s1, -c1));
        o[6] = tmul<INV>(o[6], mk<T>(-h, -h));
        o[7] = tmul<INV>(o[7], mk<T>(-c1, -s1));
        dft8<INV, false, T>(e[0], e[1], e[2], e[3], e[4], e[5], e[6], e[7]);
        dft8<INV, false, T>(o[0], o[1], o[2], o[3], o[4], o[5], o[6], o[7]);
#pragma unroll
        for (int m = 0; m < 8; ++m) { v[2 * m] = e[m]; v[2 * m + 1] = o[m]; }
    }
}

template <int LOG2LZ> struct ZCfg {
    static constexpr int LZ = 1 << LOG2LZ;
    static constexpr int LOG2E = LOG2LZ <= 3 ? LOG2LZ : (LOG2LZ + 1) / 2;
    static constexpr int E = 1 << LOG2E;          // layers per thread (registers)
    static constexpr int TT = LZ / E;             // warps per CTA
    static constexpr int RPT = E / TT;            // r values per thread after the exchange (E >= TT)
};

// STAGE: the S tile of an item ([LZ][6][32] reals, contiguous in the bank) is copied to shared memory by cp.async
// while the previous item finishes and this item's forward transform runs, so the multiply never waits for HBM
// (ncu on the register-only version: long-scoreboard stalls on the bank loads dominate).  Used where the
// exchange buffer and the tile fit together (fp32: Lz <= 128, fp64: Lz <= 64).
template <typename T, int LOG2LZ> struct ZOcc {
    typedef typename cplx_of<T>::type C;
    static constexpr int LZ = ZCfg<LOG2LZ>::LZ, TT = ZCfg<LOG2LZ>::TT;
    static constexpr int THREADS = 32 * TT;
    static constexpr size_t EX_BYTES = TT > 1 ? (size_t)3 * LZ * 32 * sizeof(C) : 0;
    static constexpr size_t BANK_BYTES = (size_t)(LZ / 2 + 1) * 6 * 32 * sizeof(T);   // kz = 0 .. LZ / 2
    static constexpr bool STAGE = TT > 1 && EX_BYTES + BANK_BYTES + LZ * sizeof(C) <= 200 * 1024;
    static constexpr size_t SMEM = EX_BYTES + (STAGE ? BANK_BYTES : 0) + LZ * sizeof(C);
};

// multiply the three components at one (k, kz) by the real symmetric S(k, kz); bt: shared or global, slot of
// min(kz, LZ - kz); neg: kz > LZ / 2, the odd components xz, yz change sign
template <bool SMEM, typename T, typename C>
__device__ __forceinline__ void zmul(const T* __restrict__ bt, bool neg, C& x, C& y, C& z) {
    T a[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) a[c] = SMEM ? bt[c * 32] : __ldcs(bt + c * 32);
    if (neg) { a[4] = -a[4]; a[5] = -a[5]; }
    const C mx = x, my = y, mz = z;
    C hx = cscale(a[0], mx), hy = cscale(a[3], mx), hz = cscale(a[4], mx);
    hx = caxpy(a[3], my, hx); hy = caxpy(a[1], my, hy); hz = caxpy(a[5], my, hz);
    hx = caxpy(a[4], mz, hx); hy = caxpy(a[5], mz, hy); hz = caxpy(a[2], mz, hz);
    x = hx; y = hy; z = hz;
}

template <typename T, int LOG2LZ>
__global__ void __launch_bounds__(ZOcc<T, LOG2LZ>::THREADS)
coupling_zfft_kernel(const T* __restrict__ bank3, HFFT_C* __restrict__ spec, const HFFT_C* __restrict__ twz, int nz,
                     int batch, long long n_tiles, long long ks) {
    typedef HFFT_C C;
    typedef ZCfg<LOG2LZ> Z;
    typedef ZOcc<T, LOG2LZ> O;
    constexpr int LZ = Z::LZ, E = Z::E, TT = Z::TT, RPT = Z::RPT, TK = 32;
    constexpr bool STAGE = O::STAGE;
    constexpr int CHUNK_T = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* ex = reinterpret_cast<C*>(smem_raw);                                   // [3][LZ][32] (TT > 1)
    T* sbank = reinterpret_cast<T*>(smem_raw + O::EX_BYTES);                   // [LZ / 2 + 1][6][32] (STAGE)
    C* stw = reinterpret_cast<C*>(smem_raw + O::EX_BYTES + (STAGE ? O::BANK_BYTES : 0));   // [LZ] exp(-2 pi i n / LZ)
    const int lane = threadIdx.x & 31, t = threadIdx.x >> 5;
    const int np = 3 * nz;
    for (int x = threadIdx.x; x < LZ; x += blockDim.x) stw[x] = twz[x];

    const long long n_items = n_tiles * batch;
    auto fetch_bank = [&](long long it) {
        if (STAGE && it < n_items) {
            const T* src = bank3 + (it / batch) * (LZ / 2 + 1) * (6LL * TK);
            for (int x = threadIdx.x; x < (LZ / 2 + 1) * 6 * TK / CHUNK_T; x += blockDim.x)
                cp_async16(sbank + x * CHUNK_T, src + x * CHUNK_T);
        }
        cp_async_commit();
    };
    fetch_bank(blockIdx.x);                                 // the S tile is constant data: it may fly before the wait
    pdl_wait();                                             // M^ comes from the previous kernel (S2)
    __syncthreads();

    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
        const long long tile = item / batch;
        const int b = (int)(item - tile * batch);
        C* sp = spec + (long long)b * np * ks + tile * TK + lane;
        C v[3][E];
        // ---- forward: DFT_E over q (upper half zero), twiddle W_LZ^{t r} ----
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int q = 0; q < E / 2; ++q) {
                const int n = t + TT * q;
                v[c][q] = n < nz ? sp[(long long)(c * nz + n) * ks] : mk<T>((T)0, (T)0);
            }
#pragma unroll
        for (int c = 0; c < 3; ++c) rdft<E, false, true, T>(v[c]);
        if constexpr (TT > 1) {
#pragma unroll
            for (int r = 1; r < E; ++r) {
                const C w = stw[(t * r) & (LZ - 1)];
#pragma unroll
                for (int c = 0; c < 3; ++c) v[c][r] = cmul(v[c][r], w);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int r = 0; r < E; ++r) ex[((c * LZ) + r * TT + t) * TK + lane] = v[c][r];
            if (STAGE) cp_async_wait_group<0>();               // this thread's part of the S tile has landed
            __syncthreads();
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr)
#pragma unroll
                    for (int s = 0; s < TT; ++s) v[c][rr * TT + s] = ex[((c * LZ) + (t * RPT + rr) * TT + s) * TK + lane];
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr) rdft<TT, false, false, T>(&v[c][rr * TT]);
        }
        // ---- v[c][rr TT + s] = M^_c(k, kz), kz = r + E s, r = t RPT + rr: multiply by S(k, kz) ----
        const T* bt = STAGE ? sbank + lane : bank3 + tile * (LZ / 2 + 1) * (6LL * TK) + lane;
#pragma unroll
        for (int rr = 0; rr < RPT; ++rr)
#pragma unroll
            for (int s = 0; s < TT; ++s) {
                const int kz = (TT > 1 ? t * RPT + rr : rr) + E * s;
                const int o = rr * TT + s;
                const bool neg = kz > LZ / 2;
                zmul<STAGE, T>(bt + (neg ? LZ - kz : kz) * 6 * TK, neg, v[0][o], v[1][o], v[2][o]);
            }
        // ---- inverse ----
        if constexpr (TT > 1) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr) rdft<TT, true, false, T>(&v[c][rr * TT]);
            __syncthreads();                                   // everyone is done with the forward exchange and the S tile
            fetch_bank(item + gridDim.x);                      // next item's S tile flies from here on
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr)
#pragma unroll
                    for (int s = 0; s < TT; ++s) ex[((c * LZ) + (t * RPT + rr) * TT + s) * TK + lane] = v[c][rr * TT + s];
            __syncthreads();
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int r = 0; r < E; ++r) v[c][r] = ex[((c * LZ) + r * TT + t) * TK + lane];
#pragma unroll
            for (int r = 1; r < E; ++r) {
                const C w = stw[(t * r) & (LZ - 1)];
#pragma unroll
                for (int c = 0; c < 3; ++c) v[c][r] = cmulc(v[c][r], w);
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            rdft<E, true, false, T>(v[c]);
#pragma unroll
            for (int q = 0; q < E / 2; ++q) {                  // crop: layers n < nz <= LZ / 2
                const int n = t + TT * q;
                if (n < nz) sp[(long long)(c * nz + n) * ks] = v[c][q];
            }
        }
        if constexpr (TT > 1) __syncthreads();                 // the exchange buffer is free again
    }
    cp_async_wait_group<0>();
}

// ---- long stacks (Lz = 128, 256; fp32): the same transform with the spectra kept in SHARED memory between the steps ----
// coupling_zfft_kernel holds all three components of a thread's layers in registers (3 x 16 complex = 96 registers at
// Lz >= 128): one 8-warp CTA per SM at Lz = 128 (ncu: 12 % warps active, latency bound at 4.2 TB/s) and spills at
// Lz = 256.  Here a thread never holds more than one 16-point transform (or three 8-point ones): the forward and the
// inverse first-stage transforms go component by component, the second-stage transform, the multiply by S(k, kz) and the
// inverse second stage work in place in the exchange buffer on the thread's own (r, all s) entries -- no extra barrier.
// Lz = 128: three 8-point transforms at a time, two CTAs per SM (measured slower than the register form, kept for A/B);
// Lz = 256 (the shipped use): 16-point transforms component by component, then the multiply four kz at a time, 16 warps
// per CTA.  The S values are read straight from global memory
// (streaming loads, 128 B per warp and value), issued ahead of the shared-memory work that hides them.
template <int LOG2LZ> struct Z2Cfg {
    static constexpr int TT = ZCfg<LOG2LZ>::TT;
    static constexpr int THREADS = 32 * TT;
    static constexpr int MINB = TT <= 8 ? 2 : 1;
    static constexpr size_t SMEM = (size_t)3 * ZCfg<LOG2LZ>::LZ * 32 * sizeof(float2) + ZCfg<LOG2LZ>::LZ * sizeof(float2);
};

template <int LOG2LZ>
__global__ void __launch_bounds__(Z2Cfg<LOG2LZ>::THREADS, Z2Cfg<LOG2LZ>::MINB)
coupling_zfft2_kernel(const float* __restrict__ bank3, float2* __restrict__ spec, const float2* __restrict__ twz, int nz,
                      int batch, long long n_tiles, long long ks) {
    typedef float T;
    typedef float2 C;
    typedef ZCfg<LOG2LZ> Z;
    constexpr int LZ = Z::LZ, E = Z::E, TT = Z::TT, RPT = Z::RPT, TK = 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* ex = reinterpret_cast<C*>(smem_raw);                                   // [3][LZ][32]
    C* stw = reinterpret_cast<C*>(smem_raw + (size_t)3 * LZ * TK * sizeof(C));  // [LZ] exp(-2 pi i n / LZ)
    const int lane = threadIdx.x & 31, t = threadIdx.x >> 5;
    const int np = 3 * nz;
    for (int x = threadIdx.x; x < LZ; x += blockDim.x) stw[x] = twz[x];
    const long long n_items = n_tiles * batch;
    pdl_wait();                                             // M^ comes from the previous kernel (S2)
    __syncthreads();

    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
        const long long tile = item / batch;
        const int b = (int)(item - tile * batch);
        C* sp = spec + (long long)b * np * ks + tile * TK + lane;
        const T* bt = bank3 + tile * (LZ / 2 + 1) * (6LL * TK) + lane;            // slots kz = 0 .. LZ / 2
        // ---- forward, first stage: DFT_E over q (upper half zero), twiddle W_LZ^{t r}; all loads first ----
        {
            C in[3][E / 2];
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int q = 0; q < E / 2; ++q) {
                    const int n = t + TT * q;
                    in[c][q] = n < nz ? sp[(long long)(c * nz + n) * ks] : mk<T>((T)0, (T)0);
                }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                C v[E];
#pragma unroll
                for (int q = 0; q < E / 2; ++q) v[q] = in[c][q];
                rdft<E, false, true, T>(v);
#pragma unroll
                for (int r = 1; r < E; ++r) v[r] = cmul(v[r], stw[(t * r) & (LZ - 1)]);
#pragma unroll
                for (int r = 0; r < E; ++r) ex[((c * LZ) + r * TT + t) * TK + lane] = v[r];
            }
        }
        __syncthreads();
        // ---- second stage, multiply, inverse second stage: in place on this thread's entries (r = t RPT + rr, all s) ----
        if constexpr (TT <= 8) {
#pragma unroll 1
            for (int rr = 0; rr < RPT; ++rr) {
                const int r = t * RPT + rr;
                constexpr int HS = TT / 2;                   // S values in two batches: 24 registers at a time
                T a[HS][6];
#pragma unroll
                for (int s = 0; s < HS; ++s) {
                    const int kz = r + E * s, kzh = kz > LZ / 2 ? LZ - kz : kz;
#pragma unroll
                    for (int c = 0; c < 6; ++c) a[s][c] = __ldcs(bt + (kzh * 6 + c) * TK);
                }
                C w[3][TT];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
#pragma unroll
                    for (int s = 0; s < TT; ++s) w[c][s] = ex[((c * LZ) + r * TT + s) * TK + lane];
                    rdft<TT, false, false, T>(w[c]);
                }
#pragma unroll
                for (int half = 0; half < 2; ++half) {
#pragma unroll
                    for (int s = 0; s < HS; ++s) {           // kz = r + E (half HS + s)
                        const int o = half * HS + s;
                        // kz > LZ / 2: S(kz) = D S(LZ - kz) D, D = diag(1, 1, -1) -- the sign goes on M_z and H_z (values
                        // already here), not on the S values still in flight
                        const T sg = (r + E * o) > LZ / 2 ? (T)-1 : (T)1;
                        const C mx = w[0][o], my = w[1][o], mz = cscale(sg, w[2][o]);
                        C hx = cscale(a[s][0], mx), hy = cscale(a[s][3], mx), hz = cscale(a[s][4], mx);
                        hx = caxpy(a[s][3], my, hx); hy = caxpy(a[s][1], my, hy); hz = caxpy(a[s][5], my, hz);
                        hx = caxpy(a[s][4], mz, hx); hy = caxpy(a[s][5], mz, hy); hz = caxpy(a[s][2], mz, hz);
                        w[0][o] = hx; w[1][o] = hy; w[2][o] = cscale(sg, hz);
                    }
                    if (half == 0) {
#pragma unroll
                        for (int s = 0; s < HS; ++s) {
                            const int kz = r + E * (HS + s), kzh = kz > LZ / 2 ? LZ - kz : kz;
#pragma unroll
                            for (int c = 0; c < 6; ++c) a[s][c] = __ldcs(bt + (kzh * 6 + c) * TK);
                        }
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    rdft<TT, true, false, T>(w[c]);
#pragma unroll
                    for (int s = 0; s < TT; ++s) ex[((c * LZ) + r * TT + s) * TK + lane] = w[c][s];
                }
            }
        } else {
            static_assert(RPT == 1 || TT <= 8, "one r per thread in the component-by-component form");
            const int r = t;
#pragma unroll 1
            for (int c = 0; c < 3; ++c) {
                C w[TT];
#pragma unroll
                for (int s = 0; s < TT; ++s) w[s] = ex[((c * LZ) + r * TT + s) * TK + lane];
                rdft<TT, false, false, T>(w);
#pragma unroll
                for (int s = 0; s < TT; ++s) ex[((c * LZ) + r * TT + s) * TK + lane] = w[s];
            }
#pragma unroll 1
            for (int s0 = 0; s0 < TT; s0 += 4) {
                T a[4][6];
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const int kz = r + E * (s0 + s), kzh = kz > LZ / 2 ? LZ - kz : kz;
#pragma unroll
                    for (int c = 0; c < 6; ++c) a[s][c] = __ldcs(bt + (kzh * 6 + c) * TK);
                }
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    C* e0 = ex + (r * TT + s0 + s) * TK + lane;
                    const T sg = (r + E * (s0 + s)) > LZ / 2 ? (T)-1 : (T)1;     // S(kz) = D S(LZ - kz) D, D = diag(1, 1, -1)
                    const C mx = e0[0], my = e0[LZ * TK], mz = cscale(sg, e0[2 * LZ * TK]);
                    C hx = cscale(a[s][0], mx), hy = cscale(a[s][3], mx), hz = cscale(a[s][4], mx);
                    hx = caxpy(a[s][3], my, hx); hy = caxpy(a[s][1], my, hy); hz = caxpy(a[s][5], my, hz);
                    hx = caxpy(a[s][4], mz, hx); hy = caxpy(a[s][5], mz, hy); hz = caxpy(a[s][2], mz, hz);
                    e0[0] = hx; e0[LZ * TK] = hy; e0[2 * LZ * TK] = cscale(sg, hz);
                }
            }
#pragma unroll 1
            for (int c = 0; c < 3; ++c) {
                C w[TT];
#pragma unroll
                for (int s = 0; s < TT; ++s) w[s] = ex[((c * LZ) + r * TT + s) * TK + lane];
                rdft<TT, true, false, T>(w);
#pragma unroll
                for (int s = 0; s < TT; ++s) ex[((c * LZ) + r * TT + s) * TK + lane] = w[s];
            }
        }
        __syncthreads();
        // ---- inverse first stage, component by component; crop to the layers n < nz <= LZ / 2 ----
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            C v[E];
#pragma unroll
            for (int r = 0; r < E; ++r) v[r] = ex[((c * LZ) + r * TT + t) * TK + lane];
#pragma unroll
            for (int r = 1; r < E; ++r) v[r] = cmulc(v[r], stw[(t * r) & (LZ - 1)]);
            rdft<E, true, false, T>(v);
#pragma unroll
            for (int q = 0; q < E / 2; ++q) {
                const int n = t + TT * q;
                if (n < nz) sp[(long long)(c * nz + n) * ks] = v[q];
            }
        }
        __syncthreads();                                     // the exchange buffer is free again
    }
}

template <int L>
static cudaError_t launch_zfft2_l(const CouplingArgs& a, cudaStream_t st) {
    auto kern = coupling_zfft2_kernel<L>;
    const size_t smem = Z2Cfg<L>::SMEM;
    static PerDevice<int> cache;
    int occ = 1;
    cudaError_t err = ctas_per_sm_cached(kern, Z2Cfg<L>::THREADS, smem, cache, occ);
    if (err != cudaSuccess) return err;
    const long long items = a.n_tiles * a.batch;
    long long grid = (long long)a.num_sms * occ;
    if (grid > items) grid = items;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(Z2Cfg<L>::THREADS), smem, st, (const float*)a.bank, (float2*)a.spec,
                      (const float2*)a.twz, a.nz, a.batch, a.n_tiles, a.ks);
}

// ---- setup: z-DFT of the Toeplitz classes ----
// cls64: [nz][6][kstride] fp64 (class d = i - j >= 0, plain layout); twz64: exp(-2 pi i n / LZ)
template <typename T>
__global__ void __launch_bounds__(128)
zdft_bank_kernel(T* __restrict__ bank3, const double* __restrict__ cls64, const double2* __restrict__ twz64, int nz,
                 int LZ, long long n_k, long long kstride, long long n_k_padded) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int kz = blockIdx.y;
    if (k >= n_k_padded) return;
    double acc[6] = {0, 0, 0, 0, 0, 0};
    if (k < n_k) {
        for (int d = 0; d < nz; ++d) {
            const double2 w = twz64[(kz * d) & (LZ - 1)];          // (cos, -sin) of 2 pi kz d / LZ
            const double wc = d == 0 ? 1.0 : 2.0 * w.x, ws = d == 0 ? 0.0 : -2.0 * w.y;
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                const double a = cls64[((size_t)d * 6 + c) * kstride + k];
                acc[c] += a * (c < 4 ? wc : ws);
            }
        }
    }
    const long long tile = k / 32;
    const int kk = (int)(k - tile * 32);
#pragma unroll
    for (int c = 0; c < 6; ++c) bank3[((tile * (LZ / 2 + 1) + kz) * 6 + c) * 32 + kk] = (T)(acc[c] / LZ);   // kz <= LZ / 2
}

cudaError_t launch_zdft_bank(void* bank3, const double* cls64, const void* twz64, int nz, int log2lz, long long n_k,
                             long long kstride, long long n_k_padded, int prec, cudaStream_t st) {
    const int LZ = 1 << log2lz;
    dim3 grid((unsigned)((n_k_padded + 127) / 128), LZ / 2 + 1);          // S(LZ - kz) = +- S(kz): kz = 0 .. LZ / 2 only
    if (prec == HFFT_F32)
        zdft_bank_kernel<float><<<grid, 128, 0, st>>>((float*)bank3, cls64, (const double2*)twz64, nz, LZ, n_k, kstride,
                                                      n_k_padded);
    else
        zdft_bank_kernel<double><<<grid, 128, 0, st>>>((double*)bank3, cls64, (const double2*)twz64, nz, LZ, n_k,
                                                       kstride, n_k_padded);
    return cudaGetLastError();
}

// fp32: Lz <= 256 (16 layers x 3 components per thread in registers); fp64: Lz <= 64
bool coupling_zfft_applies(int nz, size_t elem, int* log2lz) {
    int l = 1;
    while ((1 << l) < 2 * nz) ++l;
    if (log2lz) *log2lz = l;
    return nz >= 2 && l <= (elem == 4 ? 8 : 6);
}

template <typename T, int L>
static cudaError_t launch_zfft_l(const CouplingArgs& a, cudaStream_t st) {
    typedef HFFT_C C;
    typedef ZCfg<L> Z;
    auto kern = coupling_zfft_kernel<T, L>;
    const size_t smem = ZOcc<T, L>::SMEM;
    const int threads = 32 * Z::TT;
    static PerDevice<int> cache;
    int occ = 1;
    cudaError_t err = ctas_per_sm_cached(kern, threads, smem, cache, occ);
    if (err != cudaSuccess) return err;
    const long long items = a.n_tiles * a.batch;
    long long grid = (long long)a.num_sms * occ;
    if (grid > items) grid = items;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(threads), smem, st, (const T*)a.bank, (C*)a.spec, (const C*)a.twz, a.nz, a.batch, a.n_tiles,
                                                a.ks);
}

template <typename T>
cudaError_t launch_coupling_zfft(const CouplingArgs& a, cudaStream_t st) {
    switch (a.log2lz) {
        case 2: return launch_zfft_l<T, 2>(a, st);
        case 3: return launch_zfft_l<T, 3>(a, st);
        case 4: return launch_zfft_l<T, 4>(a, st);
        case 5: return launch_zfft_l<T, 5>(a, st);
        case 6: return launch_zfft_l<T, 6>(a, st);
        default: break;
    }
    if constexpr (sizeof(T) == 4) {
        // Lz = 128: the register-resident kernel (B200, 256 x 256 x 64: S3 0.193 ms against 0.357 ms for the shared-memory
        // form, which pays two more trips through the exchange buffer); Lz = 256: the shared-memory form (no spills:
        // evaluation 1.13 -> 0.81 ms at nz = 128, 1.02 -> 0.69 ms at nz = 96).  HFFT_ZFFT_FORM=reg|smem forces one (A/B).
        static const char* form = getenv("HFFT_ZFFT_FORM");
        const bool smem_form = form ? form[0] == 's' : a.log2lz == 8;
        if (a.log2lz == 7) return smem_form ? launch_zfft2_l<7>(a, st) : launch_zfft_l<T, 7>(a, st);
        if (a.log2lz == 8) return smem_form ? launch_zfft2_l<8>(a, st) : launch_zfft_l<T, 8>(a, st);
    }
    return cudaErrorInvalidValue;
}

template cudaError_t launch_coupling_zfft<float>(const CouplingArgs&, cudaStream_t);
template cudaError_t launch_coupling_zfft<double>(const CouplingArgs&, cudaStream_t);

}  // namespace hfft
