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

// programmatic dependent launch: wait until the preceding kernel of the stream has completed and its writes are
// visible (no-op when the kernel was not launched as a dependent)
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

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
// A bijection on [0, N) for every power of two N, and LINEAR over GF(2): swz(a ^ b) = swz(a) ^
// swz(b).  Every index used below is a sum of a per-thread part and a compile-time part that
// occupy disjoint bits, so an address is (per-thread base) XOR (compile-time constant): one
// LOP3 per shared-memory access, with the base computed once per kernel.
__host__ __device__ constexpr int swz(int i) { return i ^ ((i >> 4) & 7) ^ ((i >> 3) & 8); }

// shared-memory access by 32-bit shared-space address (the XOR arithmetic is done on integers)
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
template <typename C> __device__ __forceinline__ C lds(unsigned addr);
template <> __device__ __forceinline__ float2 lds<float2>(unsigned addr) {
    float2 v; asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory"); return v;
}
template <> __device__ __forceinline__ double2 lds<double2>(unsigned addr) {
    double2 v; asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory"); return v;
}
__device__ __forceinline__ void sts(unsigned addr, float2 v) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void sts(unsigned addr, double2 v) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}

// asynchronous 16-byte global -> shared copies (LDGSTS), bypassing L1 and the register file
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gsrc));
}
__device__ __forceinline__ void cp_async16(unsigned smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_dst), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait_group() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::: "memory");
}

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
// Everything that depends only on the thread (not on the row) lives in a Ctx that a persistent
// kernel sets up once: the twiddles of the thread's butterflies (registers if REGTW, else read
// from the thread's column of a per-thread table with immediate offsets) and the swizzled
// shared-memory base addresses.  Per row a thread then executes the butterflies, one LOP3 per
// shared-memory access and ONE barrier per exchange (two buffers per row, used alternately).
//
// Per-thread twiddle table (host: thread_twiddle_table in hfft_api.cu): for the stages after the
// first, in order, slot = OFF(stage) + u (RAD - 1) + (t - 1) holds, for thread j < TPR,
//     exp(-2 pi i t k / (N_s RAD)),  k = (j + u TPR) mod N_s,
// stored [slot][j] so that the TPR threads of a row read consecutive elements.
template <typename T, int LOG2N, bool INV, bool ZP, bool REGTW>
struct RowFFT {
    typedef HFFT_C C;
    static constexpr int N = 1 << LOG2N;
    static constexpr int LOG2R = LOG2N < 3 ? LOG2N : 3;
    static constexpr int R = 1 << LOG2R;           // elements per thread
    static constexpr int TPR = N / R;              // threads per row
    static constexpr int LOG2TPR = LOG2N - LOG2R;
    static constexpr int SH = sizeof(C) == 8 ? 3 : 4;
    static constexpr unsigned BUF_BYTES = (unsigned)N * sizeof(C);     // one exchange buffer of a row
    static constexpr unsigned ROW_BYTES = 2 * BUF_BYTES;               // a row's two buffers; rows are aligned to this

    static __host__ __device__ constexpr int lr_at(int lns) { return lns == 0 ? LOG2R : (LOG2N - lns >= 3 ? 3 : LOG2N - lns); }
    static __host__ __device__ constexpr int stages() { int n = 0; for (int l = 0; l < LOG2N; l += lr_at(l)) ++n; return n; }
    // twiddle slots used by the stages that start below lns
    static __host__ __device__ constexpr int slots_before(int lns) {
        int n = 0;
        for (int l = lr_at(0); l < lns; l += lr_at(l)) n += (R >> lr_at(l)) * ((1 << lr_at(l)) - 1);
        return n;
    }
    static constexpr int NSTAGES = stages();
    static constexpr int EXCH = NSTAGES - 1;                           // exchanges per row
    static constexpr int NSLOTS = slots_before(LOG2N);

    struct Ctx {
        C tw[NSLOTS > 0 ? NSLOTS : 1];             // REGTW only
        const C* twp;                              // twt + j
        unsigned st[NSTAGES][R];                   // st[s][u]: store base of butterfly u after stage s
        unsigned ld;                               // load base: element j of the row
        int bar, barn;                             // named barrier of the row (TPR > 32) and its thread count
    };

    // the row synchronises among its own threads only: within one warp when TPR <= 32, else on
    // the row's own named barrier (bar.sync id, TPR), so rows of a CTA never wait for each other
    static __device__ __forceinline__ void sync(const Ctx& c) {
        if (TPR <= 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(c.bar), "r"(c.barn) : "memory");
    }

    template <int LNS, int SIDX>
    static __device__ __forceinline__ void init_stage(Ctx& c, unsigned rowaddr, int j, int rx) {
        constexpr int LR = lr_at(LNS);
        if constexpr (LNS + LR < LOG2N) {
            constexpr int U = R >> LR, NS = 1 << LNS;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int b = j + u * TPR;
                const int pos = ((b >> LNS) << (LNS + LR)) + (b & (NS - 1));
                c.st[SIDX][u] = rowaddr ^ ((unsigned)(swz(pos) ^ rx) << SH);
            }
            init_stage<LNS + LR, SIDX + 1>(c, rowaddr, j, rx);
        }
    }

    // r: row slot in the CTA (at most 15 slots when TPR > 32: named barriers 1..15);
    // rowaddr: shared-space address of the row's buffer pair (ROW_BYTES aligned); rx < min(16, N)
    // is XOR-ed into every element index of the row (lets a caller read the rows "transposed",
    // lanes along rows, without bank conflicts); twt: per-thread twiddle table.
    // rpb: rows that share one named barrier (there are 15 of them: a CTA with 16 multi-warp rows pairs them up)
    static __device__ __forceinline__ void init(Ctx& c, int r, unsigned rowaddr, int j, int rx,
                                                const C* __restrict__ twt, int rpb = 1) {
        c.bar = r / rpb + 1;
        c.barn = TPR * rpb;
        c.ld = rowaddr ^ ((unsigned)(swz(j) ^ rx) << SH);
        c.twp = twt + j;
        if constexpr (REGTW) {
#pragma unroll
            for (int sl = 0; sl < NSLOTS; ++sl) c.tw[sl] = __ldg(twt + sl * TPR + j);
        }
        init_stage<0, 0>(c, rowaddr, j, rx);
    }

    // shared-space address of element (j + q TPR) of the row in buffer `par`
    template <int PAR>
    static __device__ __forceinline__ unsigned elem_addr(const Ctx& c, int q) {
        return c.ld ^ (((unsigned)swz(q * TPR) << SH) ^ (PAR ? BUF_BYTES : 0u));
    }

    template <int LNS, int SIDX, int PAR>
    static __device__ __forceinline__ void stage(C (&v)[R], const Ctx& c) {
        constexpr int LR = lr_at(LNS);
        constexpr int RAD = 1 << LR;
        constexpr int U = R / RAD;                  // butterflies per thread
        constexpr int NS = 1 << LNS;
        constexpr bool FIRST = LNS == 0;
        constexpr bool LAST = LNS + LR == LOG2N;
        constexpr int OFF = slots_before(LNS);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if constexpr (!FIRST) {
#pragma unroll
                for (int t = 1; t < RAD; ++t) {
                    const int sl = OFF + u * (RAD - 1) + (t - 1);
                    const C w = REGTW ? c.tw[sl] : __ldg(c.twp + sl * TPR);
                    v[u + t * U] = tmul<INV>(v[u + t * U], w);
                }
            }
            if constexpr (RAD == 8)
                dft8<INV, ZP && FIRST, T>(v[u], v[u + U], v[u + 2 * U], v[u + 3 * U], v[u + 4 * U], v[u + 5 * U],
                                          v[u + 6 * U], v[u + 7 * U]);
            else if constexpr (RAD == 4)
                dft4<INV, ZP && FIRST>(v[u], v[u + U], v[u + 2 * U], v[u + 3 * U]);
            else
                dft2<INV, ZP && FIRST>(v[u], v[u + U]);
        }
        if constexpr (!LAST) {
            // output t of butterfly u goes to pos(u) + t N_s; pos has zero bits where t N_s lives
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int t = 0; t < RAD; ++t)
                    sts(c.st[SIDX][u] ^ (((unsigned)swz(t * NS) << SH) ^ (PAR ? BUF_BYTES : 0u)), v[u + t * U]);
            sync(c);
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = lds<C>(elem_addr<PAR>(c, q));
            stage<LNS + LR, SIDX + 1, PAR ^ 1>(v, c);
        }
        // LAST: output t of butterfly u is X[j + (u + t U) TPR] and already sits in v[u + t U]
    }

    // v[q] = x[j + q TPR] (q < R / 2 if ZP) on entry, X[j + q TPR] on return.  Every thread of the
    // row (of the CTA if TPR > 32) must call this together.  Exchange e uses buffer e & 1, so the
    // only hazard between consecutive rows is an odd number of exchanges: one more barrier then.
    static __device__ __forceinline__ void run(C (&v)[R], const Ctx& c) {
        stage<0, 0, 0>(v, c);
        if constexpr (EXCH & 1) sync(c);
    }
};

}  // namespace hfft
