// coupling.cu -- stage S3: the explicit layer-to-layer convolution along z at every in-plane
// wavevector, the sum over j3 of Eq.24:
//
//     H^_i(k) = - sum_j N^_ij(k) M^_j(k),    N^_ij(k) a symmetric 3x3 tensor per layer pair,
//
// "the remaining convolution in the third dimension has to be calculated explicitly";
// it is the O(nz^2) term of the method.
//
// Real form: xx,yy,zz,xy spectra are purely real (A), xz,yz purely imaginary
// (i B).  With M'_z = i M_z and H'_z = i H_z the coupling is the REAL matrix
//     [Hx ; Hy ; H'z] = [[a0, a3, a4], [a3, a1, a5], [-a4, -a5, a2]] [Mx ; My ; M'z]
// acting on real and imaginary parts alike, where the bank stores, per (i, j, k),
//     a0..a5 = -s (Axx, Ayy, Azz, Axy, Bxz, Byz),  s = 1/(4 nx ny)  (sign and normalisation folded).
//
// Bank layout: [tile][i][j][6][tile_k] elements of T; one CTA item = one k-tile of one state.
// A warp owns one target layer i at a time; a lane owns KPT consecutive wavevectors, so each
// bank access of a warp is one fully coalesced 32*KPT*sizeof(T)-byte request (512 B at KPT = 4),
// and the whole [i][j][6] stream of a tile is contiguous in memory.  M^ of all layers for the
// tile sits in shared memory (cp.async, 16-byte chunks, XOR-swizzled against bank conflicts);
// H^ overwrites M^ in place (each tile is read completely before it is written).
//
// Storage variants of the same sum (each with its own kernel or template flag below):
//   mirror   (MIR)      ky and 2ny - ky share one bank entry: [tile][i][j][3 pairs][32 lanes][2], half the stream
//   recip    (CLS+MIR)  S_pq = dz_p R_pq for p <= q only, (q, p) by transposition: a quarter of the memory
//   classes  (CLS, coupling_class_kernel)  one slot per distinct (dz_i, dz_j, Z_ij); Toeplitz window for equal dz
//   batched  (coupling_batched_kernel)     B states per call, the bank of a tile held in registers
//   z-FFT    (coupling_zfft.cu)            equal dz: the z-convolution by FFT, Eq.25
#include "hfft_internal.h"
#include "fft.cuh"

namespace hfft {

// one lane's KPT consecutive bank values: streamed (evict-first: every value is used once) or, for
// the deduplicated bank, through the read-only cached path (the tile is re-read by every target layer)
template <bool CACHED, typename V> __device__ __forceinline__ V bank_ld(const V* p) {
    return CACHED ? __ldg(p) : __ldcs(p);
}
template <typename T, int KPT> struct BankVec;
template <> struct BankVec<float, 4> {
    template <bool CACHED> static __device__ __forceinline__ void ld(const float* p, float v[4]) {
        float4 t = bank_ld<CACHED>(reinterpret_cast<const float4*>(p));
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    }
};
template <> struct BankVec<float, 2> {
    template <bool CACHED> static __device__ __forceinline__ void ld(const float* p, float v[2]) {
        float2 t = bank_ld<CACHED>(reinterpret_cast<const float2*>(p));
        v[0] = t.x; v[1] = t.y;
    }
};
template <> struct BankVec<float, 1> {
    template <bool CACHED> static __device__ __forceinline__ void ld(const float* p, float v[1]) { v[0] = bank_ld<CACHED>(p); }
};
template <> struct BankVec<double, 2> {
    template <bool CACHED> static __device__ __forceinline__ void ld(const double* p, double v[2]) {
        double2 t = bank_ld<CACHED>(reinterpret_cast<const double2*>(p));
        v[0] = t.x; v[1] = t.y;
    }
};
template <> struct BankVec<double, 1> {
    template <bool CACHED> static __device__ __forceinline__ void ld(const double* p, double v[1]) { v[0] = bank_ld<CACHED>(p); }
};

// MIR (mirror layout, fft_kernels.cu ypos): the spectrum slots 2p and 2p + 1 hold ky and its mirror 2ny - ky, which
// share one bank entry p -- xx, yy, zz, xz are even in ky, xy and yz odd -- so a lane's KPT slots need
// KPT / 2 bank values per component and the odd slots take -xy, -yz: the bank stream, the only HBM-bound part, halves.
template <typename T, int KPT, bool CLS, bool MIR>
__global__ void __launch_bounds__(MIR && sizeof(T) == 4 ? 1024 : 512)
coupling_kernel(const T* __restrict__ bank, HFFT_C* __restrict__ spec, int nz, int batch, long long n_tiles,
                long long ks, int ncls, const unsigned short* __restrict__ cls, int fold, const T* __restrict__ inv_dz) {
    typedef HFFT_C C;
    static_assert(!MIR || KPT % 2 == 0, "mirror layout: an even number of slots per lane");
    // CLS && MIR = reciprocity storage (hfft_plan_set_recip): slot(i, j) = slot(j, i); the bank holds S_pq = dz_p R_pq
    // for p <= q only, the pair (q, p) uses its transpose (xz, yz negated), and H_i is scaled by 1 / dz_i at the end.
    constexpr bool RECIP = CLS && MIR;
    constexpr int TK = 32 * KPT;
    constexpr int KB = MIR ? KPT / 2 : KPT;               // bank values per lane and component
    constexpr int TKB = 32 * KB;                          // bank values per tile, pair and component
    constexpr int CHUNK_C = 16 / sizeof(C);               // complex per 16-byte chunk (2 or 1)
    constexpr int CPP = TK / CHUNK_C;                     // chunks per plane row
    constexpr bool SWZ = (KPT * sizeof(C) == 32);         // two 16-byte chunks per lane
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* sm = reinterpret_cast<C*>(smem_raw);               // [3 nz][TK] (chunk-swizzled)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int np = 3 * nz;
    const long long n_items = n_tiles * batch;
    pdl_wait();                                           // M^ comes from the previous kernel (S2)

    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
        const long long tile = item / batch;
        const int b = (int)(item - tile * batch);
        C* sp = spec + (long long)b * np * ks + tile * TK;

        for (int w = tid; w < np * CPP; w += blockDim.x) {
            const int lp = w / CPP, ch = w - lp * CPP;
            const int chs = SWZ ? (ch ^ ((ch >> 3) & 1)) : ch;
            cp_async16(sm + lp * TK + chs * CHUNK_C, sp + (long long)lp * ks + ch * CHUNK_C);
        }
        cp_async_wait_all();
        __syncthreads();

        for (int i = warp; i < nz; i += nwarps) {
            C hx[KPT], hy[KPT], hz[KPT];
#pragma unroll
            for (int e = 0; e < KPT; ++e) hx[e] = hy[e] = hz[e] = mk<T>((T)0, (T)0);
            // deduplicated bank (CLS): the slot of pair (i, j) is its tensor class; the tile is then small
            // and re-read by every target layer, so it is served from L1 / L2
            // MIR: the 6 KB values of a lane are stored as three vectors of 2 KB (component pairs (xx,yy), (zz,xy),
            // (xz,yz) x KB entries: [pair][lane][2][KB]), so that the half-width bank still moves in 16-byte loads --
            // with 8-byte loads the same bytes in flight need twice the outstanding requests and HBM idles (ncu)
            const T* bt = CLS ? bank + tile * ncls * (6LL * TKB) + lane * (MIR ? 2 * KB : KB)
                              : bank + ((tile * nz + i) * nz) * (6LL * TKB) + lane * (MIR ? 2 * KB : KB);
            // RECIP: the source layers are visited by increasing |j - i| (j = i, i+1, i-1, i+2, ...): the warps of
            // targets p and q then read the shared entry (p, q) at about the same time, so that the second read is
            // served by L2 and HBM delivers every entry once
            const int rmin = i < nz - 1 - i ? i : nz - 1 - i;
#pragma unroll (MIR ? 4 : 2)
            for (int t = 0; t < nz; ++t) {
                int j = t;
                if (RECIP) {
                    const int d = (t + 1) >> 1;
                    j = t <= 2 * rmin ? ((t & 1) ? i + d : i - d) : (i <= nz - 1 - i ? t : nz - 1 - t);
                }
                T ab[6][KB];
                const int slot = CLS ? (int)cls[i * nz + j] : j;
                if constexpr (MIR) {
#pragma unroll
                    for (int cp = 0; cp < 3; ++cp) {
                        T v2[2 * KB];
                        BankVec<T, 2 * KB>::template ld<CLS>(bt + (slot * 6 + 2 * cp) * TKB, v2);
#pragma unroll
                        for (int e = 0; e < KB; ++e) { ab[2 * cp][e] = v2[e]; ab[2 * cp + 1][e] = v2[KB + e]; }
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < 6; ++c) BankVec<T, KB>::template ld<CLS>(bt + (slot * 6 + c) * TKB, ab[c]);
                }
                // folded Toeplitz classes (fold 1): N_{-d} = N_d with xz, yz negated; reciprocity (fold 2): the pair
                // (i, j), i > j, is the transpose of the stored (j, i)
                if (CLS && ((fold == 1 && i < j) || (fold == 2 && i > j))) {
#pragma unroll
                    for (int e = 0; e < KB; ++e) { ab[4][e] = -ab[4][e]; ab[5][e] = -ab[5][e]; }
                }
                T a[6][KPT];                              // per slot; mirror slots (odd) take -xy, -yz
#pragma unroll
                for (int e = 0; e < KPT; ++e) {
                    const int eb = MIR ? e / 2 : e;
                    const bool neg = MIR && (e & 1);
                    a[0][e] = ab[0][eb]; a[1][e] = ab[1][eb]; a[2][e] = ab[2][eb]; a[4][e] = ab[4][eb];
                    a[3][e] = neg ? -ab[3][eb] : ab[3][eb];
                    a[5][e] = neg ? -ab[5][eb] : ab[5][eb];
                }
                C m[3][KPT];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const C* row = sm + (c * nz + j) * TK;
                    if (SWZ) {
                        // lane owns chunks 2*lane and 2*lane+1 of the row
                        const int c0 = 2 * lane, c1 = 2 * lane + 1;
                        const int s0 = c0 ^ ((c0 >> 3) & 1), s1 = c1 ^ ((c1 >> 3) & 1);
                        if (sizeof(T) == 4) {
                            float4 u0 = *reinterpret_cast<const float4*>(row + s0 * CHUNK_C);
                            float4 u1 = *reinterpret_cast<const float4*>(row + s1 * CHUNK_C);
                            m[c][0] = mk<T>(u0.x, u0.y); m[c][1 % KPT] = mk<T>(u0.z, u0.w);
                            m[c][2 % KPT] = mk<T>(u1.x, u1.y); m[c][3 % KPT] = mk<T>(u1.z, u1.w);
                        } else {
                            m[c][0] = row[s0 * CHUNK_C];
                            m[c][1 % KPT] = row[s1 * CHUNK_C];
                        }
                    } else if (KPT == 2 && sizeof(T) == 4) {
                        const float4 u = *reinterpret_cast<const float4*>(row + lane * 2);   // one 16-byte chunk per lane
                        m[c][0] = mk<T>(u.x, u.y); m[c][1 % KPT] = mk<T>(u.z, u.w);
                    } else {
#pragma unroll
                        for (int e = 0; e < KPT; ++e) m[c][e] = row[lane * KPT + e];
                    }
                }
#pragma unroll
                for (int e = 0; e < KPT; ++e) {
                    if (MIR) {      // twice the arithmetic per bank byte: packed FFMA2 (HFFT_MIR_PACKED experiment)
                        hx[e] = caxpy(a[0][e], m[0][e], hx[e]); hx[e] = caxpy(a[3][e], m[1][e], hx[e]); hx[e] = caxpy(a[4][e], m[2][e], hx[e]);
                        hy[e] = caxpy(a[3][e], m[0][e], hy[e]); hy[e] = caxpy(a[1][e], m[1][e], hy[e]); hy[e] = caxpy(a[5][e], m[2][e], hy[e]);
                        hz[e] = caxpy(a[2][e], m[2][e], hz[e]); hz[e] = caxpy(-a[4][e], m[0][e], hz[e]); hz[e] = caxpy(-a[5][e], m[1][e], hz[e]);
                    } else {
                    hx[e] = caxpy_s(a[0][e], m[0][e], hx[e]); hx[e] = caxpy_s(a[3][e], m[1][e], hx[e]); hx[e] = caxpy_s(a[4][e], m[2][e], hx[e]);
                    hy[e] = caxpy_s(a[3][e], m[0][e], hy[e]); hy[e] = caxpy_s(a[1][e], m[1][e], hy[e]); hy[e] = caxpy_s(a[5][e], m[2][e], hy[e]);
                    hz[e] = caxpy_s(a[2][e], m[2][e], hz[e]); hz[e] = caxpy_s(-a[4][e], m[0][e], hz[e]); hz[e] = caxpy_s(-a[5][e], m[1][e], hz[e]);
                    }
                }
            }
            if (RECIP) {
                const T sc = inv_dz[i];
#pragma unroll
                for (int e = 0; e < KPT; ++e) { hx[e] = cscale(sc, hx[e]); hy[e] = cscale(sc, hy[e]); hz[e] = cscale(sc, hz[e]); }
            }
            C* ox = sp + (long long)(0 * nz + i) * ks + lane * KPT;
            C* oy = sp + (long long)(1 * nz + i) * ks + lane * KPT;
            C* oz = sp + (long long)(2 * nz + i) * ks + lane * KPT;
            if (SWZ && sizeof(T) == 4) {
                reinterpret_cast<float4*>(ox)[0] = make_float4(hx[0].x, hx[0].y, hx[1 % KPT].x, hx[1 % KPT].y);
                reinterpret_cast<float4*>(ox)[1] = make_float4(hx[2 % KPT].x, hx[2 % KPT].y, hx[3 % KPT].x, hx[3 % KPT].y);
                reinterpret_cast<float4*>(oy)[0] = make_float4(hy[0].x, hy[0].y, hy[1 % KPT].x, hy[1 % KPT].y);
                reinterpret_cast<float4*>(oy)[1] = make_float4(hy[2 % KPT].x, hy[2 % KPT].y, hy[3 % KPT].x, hy[3 % KPT].y);
                reinterpret_cast<float4*>(oz)[0] = make_float4(hz[0].x, hz[0].y, hz[1 % KPT].x, hz[1 % KPT].y);
                reinterpret_cast<float4*>(oz)[1] = make_float4(hz[2 % KPT].x, hz[2 % KPT].y, hz[3 % KPT].x, hz[3 % KPT].y);
            } else if (KPT == 2 && sizeof(T) == 4) {
                reinterpret_cast<float4*>(ox)[0] = make_float4(hx[0].x, hx[0].y, hx[1 % KPT].x, hx[1 % KPT].y);
                reinterpret_cast<float4*>(oy)[0] = make_float4(hy[0].x, hy[0].y, hy[1 % KPT].x, hy[1 % KPT].y);
                reinterpret_cast<float4*>(oz)[0] = make_float4(hz[0].x, hz[0].y, hz[1 % KPT].x, hz[1 % KPT].y);
            } else {
#pragma unroll
                for (int e = 0; e < KPT; ++e) { ox[e] = hx[e]; oy[e] = hy[e]; oz[e] = hz[e]; }
            }
        }
        __syncthreads();   // every warp is done with the tile in shared memory
    }
}

// ------------------------------------------------------------------------------------------
// Batched mode (B magnetisation states per call, BASELINE config 5): per wavevector the coupling
// is the real (3nz x 3nz) matrix times 2B real columns.  The bank of a k-tile is read from HBM
// ONCE and kept in registers: a warp owns target layer i, a lane owns one wavevector and holds
// the 6 nz reals a^c_ij(k) of its (i, k) for all source layers j.  The states stream through a
// STAGES-deep cp.async ring of M^ tiles in shared memory ([3 nz][32] complex each); per state a
// thread does 18 nz FMAs per owned layer and writes H^ of its (i, k) in place.  A thread owns
// IPT = 2 target layers when the registers allow (nz <= 8 in fp32): M^ is then read from shared
// memory once for both (ncu: the one-layer version is shared-memory-bandwidth bound).
// Tile = 32 wavevectors (hfft_api.cu picks tile_k = 32 when this kernel applies).
// ------------------------------------------------------------------------------------------
template <typename T, int NZ, int IPT, int STAGES>
__global__ void __launch_bounds__(32 * ((NZ + IPT - 1) / IPT))
coupling_batched_kernel(const T* __restrict__ bank, HFFT_C* __restrict__ spec, int batch, long long n_tiles,
                        long long ks) {
    typedef HFFT_C C;
    constexpr int TK = 32, NP = 3 * NZ;
    constexpr int NW = (NZ + IPT - 1) / IPT;              // warps; warp w owns target layers w, w + NW, ...
    constexpr int CHUNK_C = 16 / sizeof(C);               // complex per 16-byte chunk
    constexpr int CPP = TK / CHUNK_C;                     // chunks per plane row
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* sm = reinterpret_cast<C*>(smem_raw);               // [STAGES][NP][TK]
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    pdl_wait();                                           // M^ comes from the previous kernel (S2)

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        C* sp = spec + tile * TK;
        auto issue = [&](int b) {
            if (b < batch) {
                C* dst = sm + (b % STAGES) * (NP * TK);
                const C* src = sp + (long long)b * NP * ks;
                for (int x = tid; x < NP * CPP; x += 32 * NW) {
                    const int lp = x / CPP, ch = x - lp * CPP;
                    cp_async16(dst + lp * TK + ch * CHUNK_C, src + (long long)lp * ks + ch * CHUNK_C);
                }
            }
            cp_async_commit();
        };
#pragma unroll
        for (int s = 0; s < STAGES - 1; ++s) issue(s);

        T a[IPT][NZ][6];
#pragma unroll
        for (int p = 0; p < IPT; ++p) {
            const int i = w + p * NW;
            if (i < NZ) {
                const T* bt = bank + ((tile * NZ + i) * NZ) * (6LL * TK) + lane;
#pragma unroll
                for (int j = 0; j < NZ; ++j)
#pragma unroll
                    for (int c = 0; c < 6; ++c) a[p][j][c] = __ldcs(bt + (j * 6 + c) * TK);
            }
        }

        for (int b = 0; b < batch; ++b) {
            issue(b + STAGES - 1);
            cp_async_wait_group<STAGES - 1>();
            __syncthreads();
            const C* st = sm + (b % STAGES) * (NP * TK) + lane;
            C hx[IPT], hy[IPT], hz[IPT];
#pragma unroll
            for (int p = 0; p < IPT; ++p) hx[p] = hy[p] = hz[p] = mk<T>((T)0, (T)0);
#pragma unroll
            for (int j = 0; j < NZ; ++j) {
                const C mx = st[(0 * NZ + j) * TK], my = st[(1 * NZ + j) * TK], mz = st[(2 * NZ + j) * TK];
#pragma unroll
                for (int p = 0; p < IPT; ++p) {
                    hx[p] = caxpy(a[p][j][0], mx, hx[p]); hx[p] = caxpy(a[p][j][3], my, hx[p]); hx[p] = caxpy(a[p][j][4], mz, hx[p]);
                    hy[p] = caxpy(a[p][j][3], mx, hy[p]); hy[p] = caxpy(a[p][j][1], my, hy[p]); hy[p] = caxpy(a[p][j][5], mz, hy[p]);
                    hz[p] = caxpy(a[p][j][2], mz, hz[p]); hz[p] = caxpy(-a[p][j][4], mx, hz[p]); hz[p] = caxpy(-a[p][j][5], my, hz[p]);
                }
            }
            C* o = sp + (long long)b * NP * ks + lane;
#pragma unroll
            for (int p = 0; p < IPT; ++p) {
                const int i = w + p * NW;
                if (i < NZ) {
                    o[(long long)(0 * NZ + i) * ks] = hx[p];
                    o[(long long)(1 * NZ + i) * ks] = hy[p];
                    o[(long long)(2 * NZ + i) * ks] = hz[p];
                }
            }
            __syncthreads();   // every warp is done with this stage before it is refilled
        }
        cp_async_wait_group<0>();
    }
}

// ------------------------------------------------------------------------------------------
// Deduplicated bank: layer pairs with identical (dz_i, dz_j, zeta_i - zeta_j) share
// one tensor class, bank layout [tile][class][6][32].  With few classes (equal thicknesses: 2 nz - 1
// instead of nz^2, the configuration of the paper's equidistant comparison) the
// bank of a k-tile fits in shared memory next to M^, HBM traffic drops by nz / 2, and the stage is
// bound by the FMA pipe and the shared-memory bandwidth instead.
//
// A lane owns one wavevector, a warp IPT CONSECUTIVE target layers i0 .. i0 + IPT - 1.  Per source
// layer j a thread reads M^_j(k) once (3 complex) for its IPT targets.
//  - generic classes: 6 bank reals per (i, j) from shared memory (class index from a shared table);
//  - TOEP (equal thicknesses: the tensor depends on d = i - j only; slot |d|, xz and yz negated for
//    d < 0, so the tile holds nz classes): the tensors of (i0 + p, j), p < IPT, are a sliding window
//    over d; going from j to j + 1 the window moves by one, so ONE class (6 reals) is
//    loaded per j and the other IPT - 1 stay in registers (the j loop is unrolled by IPT so that
//    the window rotates by register renaming).  Shared-memory wavefronts per j: 6 + 6 for
//    9 IPT packed FMAs -- FMA-bound at IPT = 8.
// H^ is written straight to global memory (in place of M^, whose tile was read completely first).
// ------------------------------------------------------------------------------------------
// threads per CTA = 32 * ceil(nz / IPT), nz <= kClassMaxNz
constexpr int kClassMaxNz = 96;
// (fp32: nz <= 96; fp64: nz <= 64 and its registers count double)
template <typename T, int IPT> struct ClassCfg {
    static constexpr int W = IPT * (int)sizeof(T) / 4;    // register weight of the per-thread state
    static constexpr int MAXT = W >= 8 ? (sizeof(T) == 8 ? 512 : 384) : (W == 4 ? 768 : 512);
};

// MINB = 2: two CTAs of at most 256 threads per SM (one loads its tiles while the other computes)
template <typename T, int IPT, bool TOEP, int MINB>
__global__ void __launch_bounds__(MINB == 2 ? 256 : ClassCfg<T, IPT>::MAXT, MINB)
coupling_class_kernel(const T* __restrict__ bank, HFFT_C* __restrict__ spec, const unsigned short* __restrict__ cls,
                      int nz, int ncls, int batch, long long n_tiles, long long ks) {
    typedef HFFT_C C;
    constexpr int TK = 32;
    constexpr int CHUNK_C = 16 / sizeof(C), CPP = TK / CHUNK_C;
    constexpr int CHUNK_T = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sb = reinterpret_cast<T*>(smem_raw);                                        // [ncls][6][32]
    C* sm = reinterpret_cast<C*>(smem_raw + (size_t)ncls * 6 * TK * sizeof(T));    // [3 nz][32]
    unsigned short* scls = reinterpret_cast<unsigned short*>(sm + 3 * nz * TK);    // [nz][nz] (generic)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int np = 3 * nz;
    const int i0 = warp * IPT;

    if (!TOEP) {
        for (int x = tid; x < nz * nz; x += blockDim.x) scls[x] = cls[x];
    }
    pdl_wait();                                           // M^ comes from the previous kernel (S2)
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        {
            const T* src = bank + tile * ncls * (6LL * TK);
            for (int x = tid; x < ncls * 6 * TK / CHUNK_T; x += blockDim.x)
                cp_async16(sb + x * CHUNK_T, src + x * CHUNK_T);
        }
        for (int b = 0; b < batch; ++b) {
            C* sp = spec + (long long)b * np * ks + tile * TK;
            for (int x = tid; x < np * CPP; x += blockDim.x) {
                const int lp = x / CPP, ch = x - lp * CPP;
                cp_async16(sm + lp * TK + ch * CHUNK_C, sp + (long long)lp * ks + ch * CHUNK_C);
            }
            cp_async_wait_all();
            __syncthreads();

            C hx[IPT], hy[IPT], hz[IPT];
#pragma unroll
            for (int p = 0; p < IPT; ++p) hx[p] = hy[p] = hz[p] = mk<T>((T)0, (T)0);
            T win[IPT][6];
            if (TOEP) {
#pragma unroll
                for (int p = 0; p < IPT; ++p) {
                    int c0 = i0 + p;                           // d of (i0 + p, j = 0)
                    if (c0 > ncls - 1) c0 = ncls - 1;          // layers past nz - 1 of the last warp (unused)
#pragma unroll
                    for (int c = 0; c < 6; ++c) win[p][c] = sb[(c0 * 6 + c) * TK + lane];
                }
            }
            for (int j0 = 0; j0 < nz; j0 += IPT) {
#pragma unroll
                for (int jj = 0; jj < IPT; ++jj) {
                    const int j = j0 + jj;
                    if (j < nz) {
                        const C mx = sm[(0 * nz + j) * TK + lane], my = sm[(1 * nz + j) * TK + lane],
                                mz = sm[(2 * nz + j) * TK + lane];
#pragma unroll
                        for (int p = 0; p < IPT; ++p) {
                            T a[6];
                            if (TOEP) {
#pragma unroll
                                for (int c = 0; c < 6; ++c) a[c] = win[(p - jj + IPT) % IPT][c];
                            } else {
                                int i = i0 + p;
                                if (i > nz - 1) i = nz - 1;
                                const int cl = scls[i * nz + j];
#pragma unroll
                                for (int c = 0; c < 6; ++c) a[c] = sb[(cl * 6 + c) * TK + lane];
                            }
                            hx[p] = caxpy(a[0], mx, hx[p]); hx[p] = caxpy(a[3], my, hx[p]); hx[p] = caxpy(a[4], mz, hx[p]);
                            hy[p] = caxpy(a[3], mx, hy[p]); hy[p] = caxpy(a[1], my, hy[p]); hy[p] = caxpy(a[5], mz, hy[p]);
                            hz[p] = caxpy(a[2], mz, hz[p]); hz[p] = caxpy(-a[4], mx, hz[p]); hz[p] = caxpy(-a[5], my, hz[p]);
                        }
                        if (TOEP && j + 1 < nz) {
                            // window for j + 1: targets move up one slot, the freed slot takes (i0, j + 1)
                            const int dn = i0 - j - 1;
                            const int cn = dn < 0 ? -dn : dn;
#pragma unroll
                            for (int c = 0; c < 6; ++c) {
                                const T v = sb[(cn * 6 + c) * TK + lane];
                                win[(IPT - 1 - jj) % IPT][c] = (c >= 4 && dn < 0) ? -v : v;
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int p = 0; p < IPT; ++p) {
                const int i = i0 + p;
                if (i < nz) {
                    sp[(long long)(0 * nz + i) * ks + lane] = hx[p];
                    sp[(long long)(1 * nz + i) * ks + lane] = hy[p];
                    sp[(long long)(2 * nz + i) * ks + lane] = hz[p];
                }
            }
            __syncthreads();   // every warp is done with M^ (and, after the last state, the bank) in shared memory
        }
    }
}

size_t coupling_class_smem_bytes(int nz, int n_classes, bool toeplitz, size_t elem) {
    if (nz > kClassMaxNz || (elem == 8 && nz > 64)) return (size_t)1 << 30;   // thread limits of ClassCfg
    return (size_t)n_classes * 6 * 32 * elem + (size_t)3 * nz * 32 * 2 * elem +
           (toeplitz ? 0 : (size_t)nz * nz * sizeof(unsigned short));
}

template <typename T, int IPT, bool TOEP, int MINB = 1>
static cudaError_t launch_coupling_class_t(const CouplingArgs& a, cudaStream_t st) {
    typedef HFFT_C C;
    auto kern = coupling_class_kernel<T, IPT, TOEP, MINB>;
    const size_t smem = coupling_class_smem_bytes(a.nz, a.n_classes, TOEP, sizeof(T));
    const int threads = 32 * ((a.nz + IPT - 1) / IPT);
    if (threads > (MINB == 2 ? 256 : ClassCfg<T, IPT>::MAXT)) return cudaErrorInvalidConfiguration;
    static PerDevice<int> cache;
    int nb = 1;
    cudaError_t err = ctas_per_sm_cached(kern, threads, smem, cache, nb);
    if (err != cudaSuccess) return err;
    long long grid = (long long)a.num_sms * nb;
    if (grid > a.n_tiles) grid = a.n_tiles;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(threads), smem, st, (const T*)a.bank, (C*)a.spec, a.cls, a.nz, a.n_classes, a.batch,
                                                a.n_tiles, a.ks);
}

template <typename T>
static cudaError_t launch_coupling_class(const CouplingArgs& a, cudaStream_t st) {
    // IPT target layers per warp: 8 keeps the Toeplitz window FMA-bound; fewer for thin stacks so that
    // a CTA still has several warps
    constexpr int H = sizeof(T) == 4 ? 1 : 2;             // fp64: half the layers per thread
    if (a.toeplitz) {
        if (a.nz >= 32 / H && a.nz <= 64 / H) return launch_coupling_class_t<T, 8 / H, true, 2>(a, st);
        if (a.nz >= 32 / H) return launch_coupling_class_t<T, 8 / H, true>(a, st);
        if (a.nz >= 8) return launch_coupling_class_t<T, 4 / H, true>(a, st);
        return launch_coupling_class_t<T, 1, true>(a, st);
    }
    if (a.nz >= 16) return launch_coupling_class_t<T, 4 / H, false>(a, st);
    if (a.nz >= 8) return launch_coupling_class_t<T, 2 / H, false>(a, st);
    return launch_coupling_class_t<T, 1, false>(a, st);
}

// the batched kernel keeps 6 nz reals of the bank per thread: at most 96 32-bit registers
bool coupling_batched_applies(int nz, int batch, size_t elem) {
    return batch > 1 && (size_t)6 * nz * elem <= 96 * 4;
}

template <typename T, int NZ>
static cudaError_t launch_coupling_batched_nz(const void* bank, void* spec, int batch, long long n_tiles,
                                              long long ks, int num_sms, cudaStream_t st) {
    typedef HFFT_C C;
    constexpr int STAGES = 4;
    // two target layers per thread (M^ read from shared memory once for both) while the bank
    // registers stay below ~100
    constexpr int IPT = (NZ >= 2 && 6 * NZ * 2 * sizeof(T) / 4 <= 100) ? 2 : 1;
    constexpr int THREADS = 32 * ((NZ + IPT - 1) / IPT);
    auto kern = coupling_batched_kernel<T, NZ, IPT, STAGES>;
    const size_t smem = (size_t)STAGES * 3 * NZ * 32 * sizeof(C);
    static PerDevice<int> cache;
    int occ_blocks = 1;
    cudaError_t err = ctas_per_sm_cached(kern, THREADS, smem, cache, occ_blocks);
    if (err != cudaSuccess) return err;
    long long grid = (long long)num_sms * occ_blocks;
    if (grid > n_tiles) grid = n_tiles;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(THREADS), smem, st, (const T*)bank, (C*)spec, batch, n_tiles, ks);
}

template <typename T>
static cudaError_t launch_coupling_batched(const void* bank, void* spec, int nz, int batch, long long n_tiles,
                                           long long ks, int num_sms, cudaStream_t st) {
#define HFFT_NZ_CASE(V) case V: return launch_coupling_batched_nz<T, V>(bank, spec, batch, n_tiles, ks, num_sms, st);
    switch (nz) {
        HFFT_NZ_CASE(1) HFFT_NZ_CASE(2) HFFT_NZ_CASE(3) HFFT_NZ_CASE(4) HFFT_NZ_CASE(5) HFFT_NZ_CASE(6)
        HFFT_NZ_CASE(7) HFFT_NZ_CASE(8)
        default: break;
    }
    if constexpr (sizeof(T) == 4) {
        switch (nz) {
            HFFT_NZ_CASE(9) HFFT_NZ_CASE(10) HFFT_NZ_CASE(11) HFFT_NZ_CASE(12) HFFT_NZ_CASE(13) HFFT_NZ_CASE(14)
            HFFT_NZ_CASE(15) HFFT_NZ_CASE(16)
            default: break;
        }
    }
#undef HFFT_NZ_CASE
    return cudaErrorInvalidValue;
}

size_t coupling_smem_bytes(int nz, int tile_k, size_t elem) { return (size_t)3 * nz * tile_k * 2 * elem; }

template <typename T, int KPT, bool CLS, bool MIR = false>
static cudaError_t launch_coupling_k(const CouplingArgs& a, cudaStream_t st) {
    typedef HFFT_C C;
    auto kern = coupling_kernel<T, KPT, CLS, MIR>;
    const size_t smem = coupling_smem_bytes(a.nz, 32 * KPT, sizeof(T));
    int warps = a.nz < 16 ? a.nz : 16;
    // mirror storage, many layers: the M^ tile leaves room for one CTA per SM only -- give it 32 warps (64 registers)
    // so that enough bank loads are in flight (B200, 256 x 256 x 96 fp32: 3.92 -> 2.71 ms per evaluation)
    if (MIR && sizeof(T) == 4 && smem > 113 * 1024 && a.nz >= 32) warps = 32;
    const int threads = warps * 32;
    static PerDevice<int> cache;
    int occ_blocks = 1;
    cudaError_t err = ctas_per_sm_cached(kern, threads, smem, cache, occ_blocks);
    if (err != cudaSuccess) return err;
    long long items = a.n_tiles * a.batch;
    long long grid = (long long)a.num_sms * occ_blocks;
    if (grid > items) grid = items;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(threads), smem, st, (const T*)a.bank, (C*)a.spec, a.nz, a.batch, a.n_tiles, a.ks,
                                                a.n_classes, a.cls, a.recip ? 2 : (a.toeplitz ? 1 : 0), (const T*)a.inv_dz);
}

template <typename T>
cudaError_t launch_coupling(const CouplingArgs& a, cudaStream_t st) {
    constexpr int KV = 16 / sizeof(T);
    if (a.zfft) return launch_coupling_zfft<T>(a, st);
    if (a.symv) {
        if constexpr (sizeof(T) == 4) return launch_coupling_symv(a, st);
        else return cudaErrorInvalidValue;
    }
    if (a.mirror && a.recip) return a.tile_k == 64 ? launch_coupling_k<T, 2, true, true>(a, st) : cudaErrorInvalidValue;
    if (a.cls) {
        if (a.class_kernel) return a.tile_k == 32 ? launch_coupling_class<T>(a, st) : cudaErrorInvalidValue;
        if (a.tile_k == 32 * KV) return launch_coupling_k<T, KV, true>(a, st);
        if (a.tile_k == 32) return launch_coupling_k<T, 1, true>(a, st);
        return cudaErrorInvalidValue;
    }
    if (a.mirror) return a.tile_k == 64 ? launch_coupling_k<T, 2, false, true>(a, st) : cudaErrorInvalidValue;
    if (a.tile_k == 32 && coupling_batched_applies(a.nz, a.batch, sizeof(T)))
        return launch_coupling_batched<T>(a.bank, a.spec, a.nz, a.batch, a.n_tiles, a.ks, a.num_sms, st);
    if (a.tile_k == 32 * KV) return launch_coupling_k<T, KV, false>(a, st);
    if (a.tile_k == 32) return launch_coupling_k<T, 1, false>(a, st);
    return cudaErrorInvalidValue;
}

template cudaError_t launch_coupling<float>(const CouplingArgs&, cudaStream_t);
template cudaError_t launch_coupling<double>(const CouplingArgs&, cudaStream_t);

}  // namespace hfft
