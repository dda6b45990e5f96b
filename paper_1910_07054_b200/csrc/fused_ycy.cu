// fused_ycy.cu -- stages S2 + S3 + S4 in ONE kernel: the sandwich of Eq.24
//
//     F2^-1 [ sum_{j3} N^_{i3-j3} F2(.)_{j3} ]
//
// for one kx at a time.  A CTA takes the kx column of ALL 3 nz planes: forward y transforms of the 3 nz rows of the
// transposed X^ (contiguous rows, as S2), the spectra M^(kx, ky) of all planes stay in SHARED memory, the layer
// coupling H^_i = sum_j N^_ij M^_j runs on them (plain bank layout, every value read once), the inverse y transforms (as S4, crop fused) write the column back to X^.  M^ / H^ never exist in global
// memory: two launches and 4 |M^| of traffic less per evaluation.
//
// Where it applies: two columns of 3 nz x 2ny complex (M^ and H^) plus the transform rows must fit the 227 KB of one CTA
// and there are only nx + 1 columns of work, so this is the path of the SMALL grids (BASELINE configs 1 and 2: five
// launches of a few microseconds each -> three), chosen automatically there (hfft_plan_set_fusion).  On a large grid it
// can be forced where it fits (256 x 256 x 8 fp32: 220 KB) -- measured against the staged path in
// profiles/r02_fusion.md: it loses, because it needs the plain bank (no ky-mirror / reciprocity storage: the symmetric
// matvec wants all layers of a wavevector pair in one warp and a contiguous stream per warp) and runs one CTA per SM.
//
// Coupling: M^ and H^ columns are two buffers, so the (target layer, 32-wavevector tile) tasks are independent and go
// round the warps without barriers (a lane = one wavevector).  Where the bank slice of the column (the tiles
// kx 2ny / 32 ..., contiguous in the plain bank) also fits, it is brought in by cp.async while the forward transforms
// run, so that no HBM latency is left in the coupling loop.  Real form R6 (the z planes hold i M_z / i H_z), bank
// scaled by -1 / (4 nx ny).
#include "hfft_internal.h"
#include "fft.cuh"

namespace hfft {

constexpr int kFusedThreads = 256;

template <typename T, int LOG2N, bool BANKS>
__global__ void __launch_bounds__(kFusedThreads)
fused_ycy_kernel(HFFT_C* __restrict__ xhat, const T* __restrict__ bank, int nx, int nz, int batch,
                 const HFFT_C* __restrict__ twt) {
    typedef HFFT_C C;
    typedef RowFFT<T, LOG2N, false, true, false> FF;
    typedef RowFFT<T, LOG2N, true, false, false> FI;
    constexpr int N = FF::N, R = FF::R, TPR = FF::TPR;
    constexpr int RL = R > 1 ? R / 2 : 1;                     // loads per thread forward (zero padding) = stores inverse (crop)
    constexpr int NT = N >= 32 ? N / 32 : 2;                  // bank tiles a column touches (N < 32: it may straddle two)
    extern __shared__ __align__(16) unsigned char fused_smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int r = tid >> FF::LOG2TPR, j = tid & (TPR - 1);
    const int rpc = blockDim.x >> FF::LOG2TPR;                // rows per pass
    const unsigned base = (smem_u32(fused_smem_raw) + FF::ROW_BYTES - 1) & ~(FF::ROW_BYTES - 1);
    typename FF::Ctx cf;
    typename FI::Ctx ci;
    // rows wider than a warp synchronise on named barriers 1..15: at most 15 row slots then (kFusedThreads / TPR <= 8)
    FF::init(cf, r, base + r * FF::ROW_BYTES, j, 0, twt);
    FI::init(ci, r, base + r * FF::ROW_BYTES, j, 0, twt);
    const int np = 3 * nz;
    unsigned char* after_rows = fused_smem_raw + (base - smem_u32(fused_smem_raw)) + (size_t)rpc * FF::ROW_BYTES;
    C* colm = reinterpret_cast<C*>(after_rows);               // M^ [np][N]
    C* colh = colm + (size_t)np * N;                          // H^ [np][N]
    T* sbank = reinterpret_cast<T*>(colh + (size_t)np * N);   // BANKS: [NT][nz][nz][6][32]
    const long long tile_elems = (long long)nz * nz * 6 * 32;

    for (long long item = blockIdx.x; item < (long long)(nx + 1) * batch; item += gridDim.x) {
        const int b = (int)(item / (nx + 1)), kx = (int)(item - (long long)b * (nx + 1));
        const long long k0 = (long long)kx * N, tile0 = k0 >> 5;
        if constexpr (BANKS) {                                // constant data: it may fly before the wait below
            const T* src = bank + tile0 * tile_elems;
            constexpr int CH = 16 / sizeof(T);
            for (long long x = tid; x < NT * tile_elems / CH; x += blockDim.x) cp_async16(sbank + x * CH, src + x * CH);
            cp_async_commit();
        }
        if (item == (long long)blockIdx.x) pdl_wait();        // X^ comes from the previous kernel (S1)
        C* xcol = xhat + ((long long)b * np * (nx + 1) + kx) * (N / 2);          // row of plane p: + p (nx + 1) N / 2
        // ---- S2: forward y transforms, rows -> shared column; z planes times i ----
        for (int p0 = 0; p0 < np; p0 += rpc) {
            const int p = p0 + r;
            const bool live = p < np;
            C v[R];
            const C* zin = xcol + (long long)(live ? p : 0) * (nx + 1) * (N / 2) + j;
#pragma unroll
            for (int q = 0; q < RL; ++q) v[q] = live ? zin[q * TPR] : mk<T>(0, 0);
            FF::run(v, cf);
            if (live) {
                if (p >= 2 * nz) {
#pragma unroll
                    for (int q = 0; q < R; ++q) v[q] = mul_pi(v[q]);
                }
#pragma unroll
                for (int q = 0; q < R; ++q) colm[p * N + j + q * TPR] = v[q];
            }
        }
        if constexpr (BANKS) cp_async_wait_group<0>();
        __syncthreads();
        // ---- S3: H^_i(ky) = sum_j A_ij(kx, ky) M^_j(ky); task = (32 wavevectors, target layer i) ----
        constexpr int KT = (N + 31) / 32;
        for (int task = warp; task < KT * nz; task += nwarps) {
            const int kt = task / nz, i = task - kt * nz;
            const int ky = kt * 32 + lane;
            if (ky < N) {
                const long long k = k0 + ky;
                const T* bt = (BANKS ? sbank + ((k >> 5) - tile0) * tile_elems : bank + (k >> 5) * tile_elems) +
                              (long long)i * nz * (6 * 32) + (k & 31);
                C hx = mk<T>(0, 0), hy = hx, hz = hx;
#pragma unroll 4
                for (int jj = 0; jj < nz; ++jj) {
                    T a[6];
#pragma unroll
                    for (int c = 0; c < 6; ++c) a[c] = BANKS ? bt[(jj * 6 + c) * 32] : __ldcs(bt + (jj * 6 + c) * 32);
                    const C mx = colm[jj * N + ky], my = colm[(nz + jj) * N + ky], mz = colm[(2 * nz + jj) * N + ky];
                    hx = caxpy(a[0], mx, hx); hy = caxpy(a[3], mx, hy); hz = caxpy(-a[4], mx, hz);
                    hx = caxpy(a[3], my, hx); hy = caxpy(a[1], my, hy); hz = caxpy(-a[5], my, hz);
                    hx = caxpy(a[4], mz, hx); hy = caxpy(a[5], mz, hy); hz = caxpy(a[2], mz, hz);
                }
                colh[i * N + ky] = hx; colh[(nz + i) * N + ky] = hy; colh[(2 * nz + i) * N + ky] = hz;
            }
        }
        __syncthreads();
        // ---- S4: inverse y transforms, crop to the first ny outputs; z planes times -i ----
        for (int p0 = 0; p0 < np; p0 += rpc) {
            const int p = p0 + r;
            const bool live = p < np;
            C v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = live ? colh[p * N + j + q * TPR] : mk<T>(0, 0);
            if (live && p >= 2 * nz) {
#pragma unroll
                for (int q = 0; q < R; ++q) v[q] = mul_mi(v[q]);
            }
            FI::run(v, ci);
            if (live) {
                C* dst = xcol + (long long)p * (nx + 1) * (N / 2) + j;
#pragma unroll
                for (int q = 0; q < RL; ++q) dst[q * TPR] = v[q];
            }
        }
        __syncthreads();                                      // the buffers are free for the next item
    }
}

// shared memory of the fused kernel for 2ny = 2^log2N and nz layers without / with the bank slice (0: not supported)
static size_t fused_base_bytes(int log2N, int nz, size_t elem) {
    if (log2N < 2 || log2N > 11) return 0;
    const int N = 1 << log2N, tpr = N / (log2N < 3 ? N : 8);
    if (tpr > kFusedThreads) return 0;
    const int rpc = kFusedThreads / tpr;
    if (tpr > 32 && rpc > 15) return 0;                       // named barriers 1..15
    const size_t row_bytes = (size_t)2 * N * 2 * elem;
    return (size_t)(rpc + 1) * row_bytes + (size_t)2 * 3 * nz * N * 2 * elem;
}
static size_t fused_bank_bytes(int log2N, int nz, size_t elem) {
    const int N = 1 << log2N, nt = N >= 32 ? N / 32 : 2;
    return (size_t)nt * nz * nz * 6 * 32 * elem;
}
size_t fused_ycy_smem_bytes(int log2N, int nz, size_t elem) { return fused_base_bytes(log2N, nz, elem); }
// whether the automatic mode should pick the fused kernel: only where the column's slice of the bank rides along in
// shared memory (or the column is tiny).  Measured on B200 (profiles/r02_fusion.md): with the bank read from global memory
// inside the coupling loop the kernel loses to the staged path (64 x 64 x 16: 81 vs 26 us, 128 x 128 x 8: 52 vs 30 us).
bool fused_ycy_pays(int log2N, int nz, size_t elem) {
    const size_t b = fused_base_bytes(log2N, nz, elem);
    if (b == 0) return false;
    return log2N < 5 || b + fused_bank_bytes(log2N, nz, elem) <= 222 * 1024;
}

#define FUSED_CASE(V) case V: kern = banks ? fused_ycy_kernel<T, V, true> : fused_ycy_kernel<T, V, false>; break;
template <typename T>
cudaError_t launch_fused_ycy(void* xhat, const void* bank, int nx, int log2N, int nz, int batch, const void* twt, int num_sms,
                             cudaStream_t st) {
    typedef HFFT_C C;
    size_t smem = fused_base_bytes(log2N, nz, sizeof(T));
    if (smem == 0) return cudaErrorInvalidValue;
    // the bank slice rides along where it fits; the last column's slice must not run past the bank: N < 32 columns may
    // touch a tile beyond the last one, so the slice is staged only for N >= 32
    const bool banks = log2N >= 5 && smem + fused_bank_bytes(log2N, nz, sizeof(T)) <= 222 * 1024;
    if (banks) smem += fused_bank_bytes(log2N, nz, sizeof(T));
    void (*kern)(C*, const T*, int, int, int, const C*) = nullptr;
    switch (log2N) {
        FUSED_CASE(2) FUSED_CASE(3) FUSED_CASE(4) FUSED_CASE(5) FUSED_CASE(6) FUSED_CASE(7) FUSED_CASE(8) FUSED_CASE(9)
        FUSED_CASE(10) FUSED_CASE(11)
        default: return cudaErrorInvalidValue;
    }
    static PerDevice<int> cache[2][12];
    int occ = 1;
    cudaError_t err = ctas_per_sm_cached(kern, kFusedThreads, smem, cache[banks ? 1 : 0][log2N], occ);
    if (err != cudaSuccess) return err;
    long long grid = (long long)num_sms * occ;
    const long long items = (long long)(nx + 1) * batch;
    if (grid > items) grid = items;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(kFusedThreads), smem, st, (C*)xhat, (const T*)bank, nx, nz, batch, (const C*)twt);
}
#undef FUSED_CASE

template cudaError_t launch_fused_ycy<float>(void*, const void*, int, int, int, int, const void*, int, cudaStream_t);
template cudaError_t launch_fused_ycy<double>(void*, const void*, int, int, int, int, const void*, int, cudaStream_t);

}  // namespace hfft
