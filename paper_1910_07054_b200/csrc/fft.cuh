// fft.cuh -- register-resident Stockham FFT of one contiguous row, radix 8 (+ one radix 4 / 2 stage).
//
// A row of N = 2^LOG2N complex numbers is transformed by TPR = N / R threads (R = 8, or N when
// N < 8).  Thread j holds x[j + q TPR], q < R, in registers, does the radix-R butterflies of a
// stage in registers, and exchanges data with the other threads of its row through shared
// memory between stages (autosort: natural order in, natural order out, no digit reversal).
// After the last stage thread j again holds X[j + q TPR].
//
// Stage s has radix r_s and N_s = r_0 ... r_{s-1}.  Butterfly b (0 <= b < N / r_s) reads the
// elements b + t N / r_s, t < r_s, multiplies them by exp(-+ 2 pi i t (b mod N_s) / (N_s r_s)),
// takes the r_s-point DFT and writes output t to (b div N_s) N_s r_s + (b mod N_s) + t N_s.
//
// Zero padding (the circular convolution of Eq.20-24 is made linear by padding
// nx -> 2nx, ny -> 2ny; reading A10) is implicit: with ZP the caller loads only q < R / 2 and the
// first butterfly is specialised for a zero upper half -- no zero is ever loaded or stored.
// Cropping is fused the same way: the caller of an inverse transform stores only q < R / 2, and
// the arithmetic of the unused outputs is dead code the compiler removes.
//
// Sign convention (reading A11): forward e^{-2 pi i k n / N} unnormalised, inverse e^{+...}
// unnormalised; the 1/(4 nx ny) lives in the tensor bank.
#pragma once
#include <cuda_runtime.h>

namespace hfft {

template <typename T> struct cplx_of;
template <> struct cplx_of<float> { typedef float2 type; };
template <> struct cplx_of<double> { typedef double2 type; };

template <typename T> __device__ __forceinline__ typename cplx_of<T>::type mk(T x, T y) {
    typename cplx_of<T>::type r; r.x = x; r.y = y; return r;
}
#define HFFT_C typename cplx_of<T>::type

template <typename C> __device__ __forceinline__ C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) {
    C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r;
}
// s * a and s * a + c with a real scalar s
template <typename C, typename T> __device__ __forceinline__ C cscale(T s, C a) { C r; r.x = s * a.x; r.y = s * a.y; return r; }
template <typename C, typename T> __device__ __forceinline__ C caxpy(T s, C a, C c) {
    C r; r.x = s * a.x + c.x; r.y = s * a.y + c.y; return r;
}
// scalar-instruction form for every type (two FFMA): measured faster in the streaming coupling
// kernel (B200, config 4: 2.00 ms with FFMA vs 2.39 ms with FFMA2)
template <typename C, typename T> __device__ __forceinline__ C caxpy_s(T s, C a, C c) {
    C r; r.x = s * a.x + c.x; r.y = s * a.y + c.y; return r;
}

// ---- fp32: Blackwell's packed two-lane FP32 instructions (PTX add/sub/mul/fma.f32x2, SASS FADD2 /
// FMUL2 / FFMA2).  A complex number lives in one 64-bit register pair, a complex addition is ONE
// instruction, and ptxas folds the half swaps / sign flips of multiplications by +-i and the
// broadcast of a real scalar into operand modifiers (R.F32x2.LO_HI.NP, R.F32).  The scalar FP32
// instructions issue at half rate per scheduler on sm_100, so this halves both the instruction
// count and the math-pipe time of the butterflies.  Plain (non-volatile) asm: dead outputs of the
// cropped inverse transforms are still eliminated.
__device__ __forceinline__ unsigned long long f2_bits(float2 a) { return *reinterpret_cast<unsigned long long*>(&a); }
__device__ __forceinline__ float2 bits_f2(unsigned long long a) { return *reinterpret_cast<float2*>(&a); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) {
    unsigned long long r; asm("add.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b))); return bits_f2(r);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
    unsigned long long r; asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b))); return bits_f2(r);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    unsigned long long r; asm("mul.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b))); return bits_f2(r);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)), "l"(f2_bits(c)));
    return bits_f2(r);
}
template <> __device__ __forceinline__ float2 cadd<float2>(float2 a, float2 b) { return add2(a, b); }
template <> __device__ __forceinline__ float2 csub<float2>(float2 a, float2 b) { return sub2(a, b); }
// a w = a.x (w.x, w.y) + i a.y (w.x, w.y)
template <> __device__ __forceinline__ float2 cmul<float2>(float2 a, float2 w) {
    float2 t1 = mul2(make_float2(a.x, a.x), w), t2 = mul2(make_float2(a.y, a.y), w);
    return add2(t1, make_float2(-t2.y, t2.x));
}
// a conj(w) = conj(conj(a) w): t1 = a.x w, t2 = a.y w, result (t1.x + t2.y, t2.x - t1.y)
template <> __device__ __forceinline__ float2 cmulc<float2>(float2 a, float2 w) {
    float2 t1 = mul2(make_float2(a.x, a.x), w), t2 = mul2(make_float2(a.y, a.y), w);
    return sub2(make_float2(t2.y, t2.x), make_float2(-t1.x, t1.y));
}
template <> __device__ __forceinline__ float2 cscale<float2, float>(float s, float2 a) { return mul2(make_float2(s, s), a); }
template <> __device__ __forceinline__ float2 caxpy<float2, float>(float s, float2 a, float2 c) {
    return fma2(make_float2(s, s), a, c);
}

template <typename C> __device__ __forceinline__ C mul_mi(C a) { C r; r.x = a.y; r.y = -a.x; return r; }   // -i a
template <typename C> __device__ __forceinline__ C mul_pi(C a) { C r; r.x = -a.y; r.y = a.x; return r; }   // +i a
template <typename C> __device__ __forceinline__ C cconj(C a) { C r; r.x = a.x; r.y = -a.y; return r; }
// multiplication by the stage's quarter turn: -i forward, +i inverse
template <bool INV, typename C> __device__ __forceinline__ C mul_qt(C a) { return INV ? mul_pi(a) : mul_mi(a); }
// a * w forward, a * conj(w) inverse (the tables hold exp(-2 pi i t / NT))
template <bool INV, typename C> __device__ __forceinline__ C tmul(C a, C w) { return INV ? cmulc(a, w) : cmul(a, w); }

// Shared-memory index swizzle.  Rows are accessed (a) at consecutive indices, (b) at stride 8
// (stores after the first radix-8 stage) and (c) in runs of 8 at stride 64 (stores after the
// second); XOR-ing bits 4..6 into bits 0..3 makes all three conflict free for 8-byte elements.
// A bijection on [0, N) for every power of two N.
__device__ __forceinline__ int swz(int i) { return i ^ ((i >> 4) & 7) ^ ((i >> 3) & 8); }

// ---- small DFTs in registers; ZH: the upper half of the inputs is zero (not read) ----------
template <bool INV, bool ZH, typename C> __device__ __forceinline__ void dft2(C& a0, C& a1) {
    if (ZH) { a1 = a0; return; }
    C t = a0;
    a0 = cadd(t, a1);
    a1 = csub(t, a1);
}
template <bool INV, bool ZH, typename C> __device__ __forceinline__ void dft4(C& a0, C& a1, C& a2, C& a3) {
    C t0, t1, t2, t3;
    if (ZH) { t0 = a0; t1 = a0; t2 = a1; t3 = a1; }
    else { t0 = cadd(a0, a2); t1 = csub(a0, a2); t2 = cadd(a1, a3); t3 = csub(a1, a3); }
    C q = mul_qt<INV>(t3);
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    a1 = cadd(t1, q);
    a3 = csub(t1, q);
}
// X[2m] = DFT4(a_n + a_{n+4})[m], X[2m+1] = DFT4((a_n - a_{n+4}) W_8^n)[m]
template <bool INV, bool ZH, typename T, typename C>
__device__ __forceinline__ void dft8(C& a0, C& a1, C& a2, C& a3, C& a4, C& a5, C& a6, C& a7) {
    const T h = (T)0.70710678118654752440;
    C e0, e1, e2, e3, o0, o1, o2, o3;
    if (ZH) { e0 = a0; e1 = a1; e2 = a2; e3 = a3; o0 = a0; o1 = a1; o2 = a2; o3 = a3; }
    else {
        e0 = cadd(a0, a4); e1 = cadd(a1, a5); e2 = cadd(a2, a6); e3 = cadd(a3, a7);
        o0 = csub(a0, a4); o1 = csub(a1, a5); o2 = csub(a2, a6); o3 = csub(a3, a7);
    }
    // o1 *= W8, o2 *= W8^2, o3 *= W8^3 with W8 = exp(-+ i pi / 4)
    // W8 a = h (a - i a), W8^3 a = -h (a + i a) forward; conjugates inverse
    if (!INV) {
        o1 = cscale(h, cadd(o1, mul_mi(o1)));
        o2 = mul_mi(o2);
        o3 = cscale(-h, csub(o3, mul_mi(o3)));
    } else {
        o1 = cscale(h, cadd(o1, mul_pi(o1)));
        o2 = mul_pi(o2);
        o3 = cscale(-h, csub(o3, mul_pi(o3)));
    }
    dft4<INV, false>(e0, e1, e2, e3);
    dft4<INV, false>(o0, o1, o2, o3);
    a0 = e0; a1 = o0; a2 = e1; a3 = o1; a4 = e2; a5 = o2; a6 = e3; a7 = o3;
}

// ---- the row transform ------------------------------------------------------------------------
template <typename T, int LOG2N, bool INV, bool ZP>
struct RowFFT {
    typedef HFFT_C C;
    static constexpr int N = 1 << LOG2N;
    static constexpr int LOG2R = LOG2N < 3 ? LOG2N : 3;
    static constexpr int R = 1 << LOG2R;           // elements per thread
    static constexpr int TPR = N / R;              // threads per row
    static constexpr int LOG2TPR = LOG2N - LOG2R;

    // twiddles of one butterfly: w[t] = tw[t k step], t = 1 .. RAD-1 (k step < NT / RAD)
    template <int RAD>
    static __device__ __forceinline__ void twiddles(C (&w)[8], const C* __restrict__ tw, int idx) {
        w[1] = __ldg(tw + idx);
        if (RAD >= 4) { w[2] = __ldg(tw + 2 * idx); w[3] = __ldg(tw + 3 * idx); }
        if (RAD >= 8) {
            w[4] = __ldg(tw + 4 * idx); w[5] = __ldg(tw + 5 * idx);
            w[6] = __ldg(tw + 6 * idx); w[7] = __ldg(tw + 7 * idx);
        }
    }

    // One stage of radix 2^LR at N_s = 2^LNS, followed (unless it is the last) by the exchange.
    template <int LNS, int LR>
    static __device__ __forceinline__ void stage(C (&v)[R], C* __restrict__ srow, int j, const C* __restrict__ tw,
                                                 int twmul) {
        constexpr int RAD = 1 << LR;
        constexpr int U = R / RAD;                  // butterflies per thread
        constexpr int NS = 1 << LNS;
        constexpr bool FIRST = LNS == 0;
        constexpr bool LAST = LNS + LR == LOG2N;
        int pos[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int b = j + u * TPR;
            const int k = b & (NS - 1);
            if constexpr (!FIRST) {
                C w[8];
                twiddles<RAD>(w, tw, k * ((N >> (LNS + LR)) * twmul));
#pragma unroll
                for (int t = 1; t < RAD; ++t) v[u + t * U] = tmul<INV>(v[u + t * U], w[t]);
            }
            if constexpr (RAD == 8)
                dft8<INV, ZP && FIRST, T>(v[u], v[u + U], v[u + 2 * U], v[u + 3 * U], v[u + 4 * U], v[u + 5 * U],
                                          v[u + 6 * U], v[u + 7 * U]);
            else if constexpr (RAD == 4)
                dft4<INV, ZP && FIRST>(v[u], v[u + U], v[u + 2 * U], v[u + 3 * U]);
            else
                dft2<INV, ZP && FIRST>(v[u], v[u + U]);
            pos[u] = ((b >> LNS) << (LNS + LR)) + k;
        }
        if constexpr (!LAST) {
            __syncthreads();                        // earlier readers of the row are done
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int t = 0; t < RAD; ++t) srow[swz(pos[u] + t * NS)] = v[u + t * U];
            __syncthreads();
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = srow[swz(j + q * TPR)];
            constexpr int LEFT = LOG2N - LNS - LR;  // > 0 here
            constexpr int NLR = LEFT >= 3 ? 3 : LEFT;
            stage<LNS + LR, NLR>(v, srow, j, tw, twmul);
        }
        // LAST: output t of butterfly u is X[j + (u + t U) TPR] and already sits in v[u + t U]
    }

    // v[q] = x[j + q TPR] (q < R / 2 if ZP) on entry, X[j + q TPR] on return.  Every thread of the
    // CTA must call this together (it contains __syncthreads); srow is this row's N-element buffer.
    static __device__ __forceinline__ void run(C (&v)[R], C* __restrict__ srow, int j, const C* __restrict__ tw,
                                               int twmul) {
        stage<0, LOG2R>(v, srow, j, tw, twmul);
    }
};

}  // namespace hfft
