// subfft.cuh -- the transform engine of the hot-path FFT kernels (fft_hot.cu): a FULL complex FFT of M = 2^LOG2M points
// held 16 (fp32) or 8 (fp64) elements per thread, radix 16 / 8 in registers, Stockham autosort through shared memory.
//
// Why half-length transforms.  Every transform of the hot path is either zero-padded (forward: the upper half of the
// 2M inputs is zero, PAPER.md:159-178 / reading A10) or cropped (inverse: only the first M of the 2M outputs are kept).
// One radix-2 decimation-in-frequency step makes both trivial and leaves two INDEPENDENT M-point transforms:
//
//   forward, x[n] = 0 for n >= M:     X[2k]   = DFT_M(x[n])[k]                    X[2k+1] = DFT_M(x[n] w_2M^n)[k]
//   inverse, outputs n < M only:      z[2n']  = IDFT_M(X[k] + X[k+M])[n']         z[2n'+1] = IDFT_M((X[k] - X[k+M]) w_2M^-k)[n']
//                                     (n' < M / 2: the upper half of each sub-transform's outputs is dead code)
//
// so a row of 2M points costs two M-point transforms: half the shared-memory exchange traffic of a 2M-point transform
// whose first butterfly merely knows about the zeros (fft.cuh, RowFFT), and with 16 elements per thread one exchange
// less again (M = 256: 16 x 16, ONE exchange; M = 512: 16 x 16 x 2).  The two sub-transforms (h = 0: even, h = 1: odd
// outputs) belong to two groups of TPR = M / R threads; a group never spans more than one warp for M <= 512 (fp32), so
// its exchanges synchronise with __syncwarp only.
//
// Thread j of a group holds x[j + q TPR], q < R, on entry and X[j + q TPR] on return (natural order, no digit reversal).
// Stage s has radix r_s (R for every stage but possibly the last) and N_s = r_0 ... r_{s-1}; butterfly b reads the
// elements b + t M / r_s, multiplies them by exp(-+ 2 pi i t (b mod N_s) / (N_s r_s)), takes the r_s-point DFT and writes
// output t to (b div N_s) N_s r_s + (b mod N_s) + t N_s.
//
// Twiddles (host: sub_twiddle_table in hfft_api.cu).  Middle stages (radix R, one butterfly per thread): slot t - 1
// holds exp(-2 pi i t (j mod N_s) / (N_s R)) for thread j.  Last stage with radix r < R (U = R / r butterflies per
// thread, b = j + u TPR, N_s = M / r so that b mod N_s = b): only the r - 1 "bases" exp(-2 pi i t j / M) are stored; the
// factor exp(-2 pi i t u / R) that butterfly u adds is a compile-time R-th root of unity.  Slots are stored [slot][j];
// with REGTW the thread keeps its column in registers for the whole (persistent) kernel.
#pragma once
#include <type_traits>

#include "fft.cuh"

namespace hfft {

// compile-time loop: f(std::integral_constant<int, I>) for I = 0 .. N - 1 (indices usable as template arguments)
template <int I, int N, typename F> __device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// cos(2 pi n / 64), n = 0..16: every root of unity the kernels need as a compile-time constant (R-th, 2R-th and 4R-th
// roots for R <= 16) is one of the 64th roots
__host__ __device__ constexpr double cos64_q(int n) {
    constexpr double c[17] = {1.0,
                              0.99518472667219688624, 0.98078528040323044913, 0.95694033573220886494,
                              0.92387953251128675613, 0.88192126434835502971, 0.83146961230254523708,
                              0.77301045336273696081, 0.70710678118654752440, 0.63439328416364549822,
                              0.55557023301960222474, 0.47139673682599764856, 0.38268343236508977173,
                              0.29028467725446236764, 0.19509032201612826785, 0.09801714032956060199, 0.0};
    return c[n];
}
__host__ __device__ constexpr double cos64(int n) {       // cos(2 pi n / 64), any n
    n = ((n % 64) + 64) % 64;
    return n <= 16 ? cos64_q(n) : (n <= 32 ? -cos64_q(32 - n) : (n <= 48 ? -cos64_q(n - 32) : cos64_q(64 - n)));
}
__host__ __device__ constexpr double sin64(int n) { return cos64(n - 16); }

// a * exp(-2 pi i NUM / 64)  (CONJ: a * exp(+2 pi i NUM / 64)); the constant folds into immediates
template <int NUM, bool CONJ, typename C> __device__ __forceinline__ C mul_root64(C a) {
    constexpr int n = ((NUM % 64) + 64) % 64;
    if constexpr (n == 0) return a;
    else if constexpr (n == 32) { C r; r.x = -a.x; r.y = -a.y; return r; }
    else if constexpr (n == 16) return CONJ ? mul_pi(a) : mul_mi(a);
    else if constexpr (n == 48) return CONJ ? mul_mi(a) : mul_pi(a);
    else {
        typedef decltype(a.x) T;
        constexpr T cr = (T)cos64(n), si = (T)(CONJ ? sin64(n) : -sin64(n));   // w = cr + i si
        C r;
        r.x = a.x * cr - a.y * si;
        r.y = a.x * si + a.y * cr;
        return r;
    }
}

// 16-point DFT in registers as 4 x 4: n = 4 a + b, k = c + 4 d,
//   X[c + 4 d] = sum_b W4^{b d} [ W16^{b c} sum_a W4^{a c} x[4 a + b] ]
// ZH: the inputs 8..15 are zero (not read).
template <bool INV, bool ZH, typename T, typename C> __device__ __forceinline__ void dft16(C (&v)[16]) {
#pragma unroll
    for (int b = 0; b < 4; ++b) dft4<INV, ZH>(v[b], v[b + 4], v[b + 8], v[b + 12]);       // v[b + 4 c] = y_b[c]
    // twiddles W16^{b c} = exp(-+ 2 pi i 4 b c / 64)
    v[5] = mul_root64<4, INV>(v[5]);   v[9] = mul_root64<8, INV>(v[9]);    v[13] = mul_root64<12, INV>(v[13]);
    v[6] = mul_root64<8, INV>(v[6]);   v[10] = mul_root64<16, INV>(v[10]); v[14] = mul_root64<24, INV>(v[14]);
    v[7] = mul_root64<12, INV>(v[7]);  v[11] = mul_root64<24, INV>(v[11]); v[15] = mul_root64<36, INV>(v[15]);
#pragma unroll
    for (int c = 0; c < 4; ++c) dft4<INV, false>(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);   // v[4 c + d] = X[c + 4 d]
    C t;
#define HFFT_SWAP(a, b) t = v[a]; v[a] = v[b]; v[b] = t;
    HFFT_SWAP(1, 4) HFFT_SWAP(2, 8) HFFT_SWAP(3, 12) HFFT_SWAP(6, 9) HFFT_SWAP(7, 13) HFFT_SWAP(11, 14)
#undef HFFT_SWAP
}

template <typename T, int LOG2M, bool INV, int LOG2RMAX, bool REGTW>
struct SubFFT {
    typedef HFFT_C C;
    static constexpr int M = 1 << LOG2M;
    static constexpr int LOG2R = LOG2M < LOG2RMAX ? LOG2M : LOG2RMAX;
    static constexpr int R = 1 << LOG2R;           // elements per thread
    static constexpr int TPR = M / R;              // threads per sub-transform
    static constexpr int LOG2TPR = LOG2M - LOG2R;
    static constexpr int SH = sizeof(C) == 8 ? 3 : 4;
    static constexpr unsigned SUB_BYTES = (unsigned)M * sizeof(C);     // exchange buffer of a sub-transform (aligned to this)

    static __host__ __device__ constexpr int lr_at(int lns) { return LOG2M - lns >= LOG2R ? LOG2R : LOG2M - lns; }
    static __host__ __device__ constexpr int stages() { int n = 0; for (int l = 0; l < LOG2M; l += lr_at(l)) ++n; return n; }
    static __host__ __device__ constexpr int slots_before(int lns) {
        int n = 0;
        for (int l = lr_at(0); l < lns; l += lr_at(l)) n += (1 << lr_at(l)) - 1;
        return n;
    }
    static constexpr int NSTAGES = LOG2M == 0 ? 1 : stages();
    static constexpr int EXCH = NSTAGES - 1;
    static constexpr int NSLOTS = slots_before(LOG2M);

    // XOR-linear index swizzle: the stride-R stores after the first stage, the stride-R^2 runs after the second and
    // the consecutive loads are all conflict free (16 lanes x 8 bytes or 8 lanes x 16 bytes per wavefront)
    static __host__ __device__ constexpr int swz(int i) { return i ^ ((i >> LOG2R) & (R - 1)); }

    struct Ctx {
        C tw[NSLOTS > 0 ? NSLOTS : 1];             // REGTW only
        const C* twp;                              // table + j
        unsigned st[NSTAGES][R];                   // st[s][u]: store base of butterfly u after stage s
        unsigned ld;                               // load base: element j
    };

    static __device__ __forceinline__ void sync() {
        if (TPR <= 32) __syncwarp();
        else __syncthreads();                      // callers with TPR > 32 keep every thread of the CTA in step
    }

    template <int LNS, int SIDX>
    static __device__ __forceinline__ void init_stage(Ctx& c, unsigned sub, int j) {
        constexpr int LR = lr_at(LNS);
        if constexpr (LNS + LR < LOG2M) {
            constexpr int U = R >> LR, NS = 1 << LNS;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int b = j + u * TPR;
                const int pos = ((b >> LNS) << (LNS + LR)) + (b & (NS - 1));
                c.st[SIDX][u] = sub ^ ((unsigned)swz(pos) << SH);
            }
            init_stage<LNS + LR, SIDX + 1>(c, sub, j);
        }
    }

    // sub: shared-space address of the sub-transform's buffer pair (SUB_BYTES aligned); twt: the twiddle table
    static __device__ __forceinline__ void init(Ctx& c, unsigned sub, int j, const C* __restrict__ twt) {
        c.ld = sub ^ ((unsigned)swz(j) << SH);
        c.twp = twt + j;
        if constexpr (REGTW) {
#pragma unroll
            for (int sl = 0; sl < NSLOTS; ++sl) c.tw[sl] = __ldg(twt + sl * TPR + j);
        }
        if constexpr (LOG2M > 0) init_stage<0, 0>(c, sub, j);
    }

    template <int LNS, int SIDX>
    static __device__ __forceinline__ void stage(C (&v)[R], const Ctx& c) {
        constexpr int LR = lr_at(LNS);
        constexpr int RAD = 1 << LR;
        constexpr int U = R / RAD;                  // butterflies per thread (> 1 only in a last stage of radix < R)
        constexpr int NS = 1 << LNS;
        constexpr bool FIRST = LNS == 0;
        constexpr bool LAST = LNS + LR == LOG2M;
        constexpr int OFF = slots_before(LNS);
        static_assert(U == 1 || LAST, "a stage of radix < R must be the last one");
        if constexpr (!FIRST) {
            static_for<1, RAD>([&](auto tc) {
                constexpr int t = decltype(tc)::value;
                const C w = REGTW ? c.tw[OFF + t - 1] : __ldg(c.twp + (OFF + t - 1) * TPR);
                static_for<0, U>([&](auto uc) {
                    constexpr int u = decltype(uc)::value;
                    // butterfly u: exp(-2 pi i t (j + u TPR) / M) = base_t * exp(-2 pi i t u / R)
                    v[u + t * U] = mul_root64<t * u * (64 / R), INV>(tmul<INV>(v[u + t * U], w));
                });
            });
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if constexpr (RAD == 16) dft16<INV, false, T>(v);
            else if constexpr (RAD == 8)
                dft8<INV, false, T>(v[u], v[u + U], v[u + 2 * U], v[u + 3 * U], v[u + 4 * U], v[u + 5 * U], v[u + 6 * U], v[u + 7 * U]);
            else if constexpr (RAD == 4) dft4<INV, false>(v[u], v[u + U], v[u + 2 * U], v[u + 3 * U]);
            else if constexpr (RAD == 2) dft2<INV, false>(v[u], v[u + U]);
        }
        if constexpr (!LAST) {
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int t = 0; t < RAD; ++t)
                    sts(c.st[SIDX][u] ^ ((unsigned)swz(t * NS) << SH), v[u + t * U]);
            sync();
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = lds<C>(c.ld ^ ((unsigned)swz(q * TPR) << SH));
            sync();                                 // the buffer is free for the next exchange (of this or the next transform)
            stage<LNS + LR, SIDX + 1>(v, c);
        }
    }

    // v[q] = x[j + q TPR] on entry, X[j + q TPR] on return.  One buffer per sub-transform: an exchange is store,
    // synchronise, load, synchronise (warp-level for TPR <= 32).
    static __device__ __forceinline__ void run(C (&v)[R], const Ctx& c) {
        if constexpr (LOG2M > 0) stage<0, 0>(v, c);
    }
};

}  // namespace hfft
