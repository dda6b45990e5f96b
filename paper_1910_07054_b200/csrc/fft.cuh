// fft.cuh -- shared-memory radix-4 (+ one radix-2) FFT building blocks.
//
// Forward transforms are decimation-in-frequency: natural order in, digit-reversed order out,
// in place in shared memory.  Inverse transforms are decimation-in-time on digit-reversed
// input: natural order out.  Neither needs a reordering pass because the global-memory
// load / store of each kernel applies the digit permutation row by row.
//
// Zero padding (the circular convolution of Eq.20-24 is made linear by
// padding nx -> 2nx, ny -> 2ny; reading A10) is implicit: the first radix-4 stage of a forward
// transform reads only the two non-zero quarters of its input straight from global memory.
// Cropping is fused the same way: the last radix-4 stage of an inverse transform computes only
// the first half of its outputs and writes them straight to global memory.
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
template <typename C> __device__ __forceinline__ C mul_mi(C a) { C r; r.x = a.y; r.y = -a.x; return r; }   // -i a
template <typename C> __device__ __forceinline__ C mul_pi(C a) { C r; r.x = -a.y; r.y = a.x; return r; }   // +i a
template <typename C> __device__ __forceinline__ C cconj(C a) { C r; r.x = a.x; r.y = -a.y; return r; }

// ---- digit permutation of the radix-(4,...,4[,2]) DIF --------------------------------------
// reverse the order of S two-bit groups
__device__ __forceinline__ unsigned rev_groups(unsigned q, int S) {
    if (S == 0) return 0u;
    unsigned r = __brev(q) >> (32 - 2 * S);
    return ((r & 0x55555555u) << 1) | ((r >> 1) & 0x55555555u);
}
// frequency held at position p after the forward DIF
template <int LOG2N> __device__ __forceinline__ int pos2freq(int p) {
    constexpr int S = LOG2N / 2;
    if (LOG2N & 1) return (int)(((unsigned)(p & 1) << (2 * S)) | rev_groups((unsigned)p >> 1, S));
    return (int)rev_groups((unsigned)p, S);
}
// position at which frequency k sits
template <int LOG2N> __device__ __forceinline__ int freq2pos(int k) {
    constexpr int S = LOG2N / 2;
    if (LOG2N & 1) return (int)((rev_groups((unsigned)k & ((1u << (2 * S)) - 1u), S) << 1) | ((unsigned)k >> (2 * S)));
    return (int)rev_groups((unsigned)k, S);
}

// ---- radix-4 butterflies -------------------------------------------------------------------
// forward DIF: y_m = (sum_r a_r (-i)^{rm}) * W^{jm}; caller applies the twiddles
template <typename C> __device__ __forceinline__ void bfly4_fwd(C& a0, C& a1, C& a2, C& a3) {
    C t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = csub(a1, a3);
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    C mt3 = mul_mi(t3);
    a1 = cadd(t1, mt3);
    a3 = csub(t1, mt3);
}
// inverse DIT: y_r = sum_m b_m (+i)^{rm}
template <typename C> __device__ __forceinline__ void bfly4_inv(C& b0, C& b1, C& b2, C& b3) {
    C t0 = cadd(b0, b2), t1 = csub(b0, b2), t2 = cadd(b1, b3), t3 = csub(b1, b3);
    b0 = cadd(t0, t2);
    b2 = csub(t0, t2);
    C pt3 = mul_pi(t3);
    b1 = cadd(t1, pt3);
    b3 = csub(t1, pt3);
}

// Twiddle table: tw[t] = exp(-2 pi i t / NT), t in [0, NT).  A transform of length N <= NT that
// divides NT uses stride NT / N.
template <typename C> __device__ __forceinline__ C ldtw(const C* __restrict__ tw, int idx) { return __ldg(tw + idx); }

// One in-place forward DIF radix-4 stage on block length L (Q = L / 4) for butterfly t of one
// sequence whose element e lives at s[e * ES]; twiddle W_L^{jm} = tw[j m twmul].
template <typename C>
__device__ __forceinline__ void dif4_stage(C* s, const int ES, int t, int log2Q, const C* __restrict__ tw, int twmul) {
    const int Q = 1 << log2Q;
    const int j = t & (Q - 1);
    const int base = ((t >> log2Q) << (log2Q + 2)) + j;
    C a0 = s[(base) * ES], a1 = s[(base + Q) * ES], a2 = s[(base + 2 * Q) * ES], a3 = s[(base + 3 * Q) * ES];
    bfly4_fwd(a0, a1, a2, a3);
    if (log2Q > 0) {     // Q == 1: j == 0, twiddles are 1
        const int w = j * twmul;
        a1 = cmul(a1, ldtw(tw, w));
        a2 = cmul(a2, ldtw(tw, 2 * w));
        a3 = cmul(a3, ldtw(tw, 3 * w));
    }
    s[(base) * ES] = a0; s[(base + Q) * ES] = a1; s[(base + 2 * Q) * ES] = a2; s[(base + 3 * Q) * ES] = a3;
}
// One in-place inverse DIT radix-4 stage (conjugate twiddles first, then butterfly).
template <typename C>
__device__ __forceinline__ void dit4_stage(C* s, const int ES, int t, int log2Q, const C* __restrict__ tw, int twmul) {
    const int Q = 1 << log2Q;
    const int j = t & (Q - 1);
    const int base = ((t >> log2Q) << (log2Q + 2)) + j;
    C b0 = s[(base) * ES], b1 = s[(base + Q) * ES], b2 = s[(base + 2 * Q) * ES], b3 = s[(base + 3 * Q) * ES];
    if (log2Q > 0) {
        const int w = j * twmul;
        b1 = cmulc(b1, ldtw(tw, w));
        b2 = cmulc(b2, ldtw(tw, 2 * w));
        b3 = cmulc(b3, ldtw(tw, 3 * w));
    }
    bfly4_inv(b0, b1, b2, b3);
    s[(base) * ES] = b0; s[(base + Q) * ES] = b1; s[(base + 2 * Q) * ES] = b2; s[(base + 3 * Q) * ES] = b3;
}
// radix-2 stage on blocks of length 2 (no twiddles): butterfly t touches elements 2t, 2t+1
template <typename C> __device__ __forceinline__ void r2_stage(C* s, const int ES, int t) {
    C a0 = s[(2 * t) * ES], a1 = s[(2 * t + 1) * ES];
    s[(2 * t) * ES] = cadd(a0, a1);
    s[(2 * t + 1) * ES] = csub(a0, a1);
}

}  // namespace hfft
