// coupling_symv.cu -- stage S3 on the reciprocity bank: the layer-to-layer convolution of Eq.24,
//
//     H^_i(k) = - sum_j N^_ij(k) M^_j(k),
//
// with every 3 x 3 block of the bank read from HBM ONCE and used for both layer pairs it serves (layout, schedule and
// the symmetry behind it: symv_layout.h).  The O(nz^2) stream of PAPER.md:189 is a quarter of the plain real bank.
//
// Work distribution.  A warp owns EPW bank entries (= wavevector pairs ky, 2ny - ky) for ALL layers: lane = (entry, strip
// w of four layers, mirror slot s).  A lane keeps M^ and the H^ accumulators of its four layers in registers (complex:
// packed FFMA2 on (re, im) with the real bank value broadcast).  At step T it multiplies its block (w, w + T): the source
// values M^_q come from the lane that owns strip w + T by warp shuffle, the transposed contributions S^T M^_p go back to
// that lane by warp shuffle -- no shared-memory traffic for M^ / H^ in the loop and no barrier: the warps of a CTA run
// independently.  The diagonal and the half block need no exchange beyond that (symv_layout.h).
//
// Bank stream.  The unit's stream is contiguous (NC couples of 768 B).  Each warp runs its own ring of NS stages of four
// couples (3 KB; the last stage of a unit is a single couple) in shared memory, filled by bulk asynchronous copies (cp.async.bulk, the TMA engine; SASS UBLKCP) that signal an
// mbarrier per stage, with an L2 evict-first policy (every bank byte is used once); lane 0 re-arms a stage as soon as
// the warp has consumed it, across unit boundaries, so the stream never drains between tiles.  The 16 strip-lanes read a
// stage with 128-bit shared loads (the two mirror-slot lanes of a strip read the same address: broadcast).
//
// M^ / H^ tile.  A CTA of NWARP warps handles TE = NWARP EPW consecutive entries: the [3 nz][2 TE] slots of M^ come in
// by cp.async (rows of 16 TE bytes) ONE ITEM AHEAD into the other of two tile buffers, every lane picks up its own 12
// values, and H^ goes back through the same shared tile (each lane overwrites exactly the slots it read) and out in
// full rows.
#include <stdint.h>

#include "hfft_internal.h"
#include "fft.cuh"
#include "symv_layout.h"

namespace hfft {

namespace {

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ uint64_t evict_first_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// bulk asynchronous copy global -> shared (TMA engine), completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float fxor(float a, uint32_t m) { return __uint_as_float(__float_as_uint(a) ^ m); }
__device__ __forceinline__ float2 shfl2(float2 v, int src) {
    float2 r;
    r.x = __shfl_sync(0xffffffffu, v.x, src);
    r.y = __shfl_sync(0xffffffffu, v.y, src);
    return r;
}

// two pairs of a strip-lane: 12 floats in three 128-bit registers
struct Couple {
    float4 v[3];
    __device__ __forceinline__ void load(uint32_t addr) {
#pragma unroll
        for (int j = 0; j < 3; ++j) v[j] = lds128(addr + 256 * j);
    }
    // pair h (0 / 1) as a0..a5 = (xx, yy, zz, xy, xz, yz); tm flips xz, yz (transpose).  The sign change of xy, yz on the
    // mirror wavevector 2ny - ky is NOT applied here: A' = D A D with D = diag(1, -1, 1), so the odd-slot lanes work on
    // D M^ and produce D H^ with the stored block as it is (the y components are negated once per tile, on the way
    // in and on the way out, instead of two sign flips per block).
    template <int H>
    __device__ __forceinline__ void get(float (&a)[6]) const {
        if (H == 0) { a[0] = v[0].x; a[1] = v[0].y; a[2] = v[0].z; a[3] = v[0].w; a[4] = v[1].x; a[5] = v[1].y; }
        else        { a[0] = v[1].z; a[1] = v[1].w; a[2] = v[2].x; a[3] = v[2].y; a[4] = v[2].z; a[5] = v[2].w; }
    }
    template <int H>
    __device__ __forceinline__ void get(float (&a)[6], uint32_t tm) const {
        get<H>(a);
        a[4] = fxor(a[4], tm);
        a[5] = fxor(a[5], tm);
    }
};

// h += A m, A = [[a0, a3, a4], [a3, a1, a5], [-a4, -a5, a2]]  (real form R6; coupling.cu)
__device__ __forceinline__ void mv(float2 (&h)[3], const float (&a)[6], const float2 (&m)[3]) {
    h[0] = caxpy(a[0], m[0], h[0]); h[1] = caxpy(a[3], m[0], h[1]); h[2] = caxpy(-a[4], m[0], h[2]);
    h[0] = caxpy(a[3], m[1], h[0]); h[1] = caxpy(a[1], m[1], h[1]); h[2] = caxpy(-a[5], m[1], h[2]);
    h[0] = caxpy(a[4], m[2], h[0]); h[1] = caxpy(a[5], m[2], h[1]); h[2] = caxpy(a[2], m[2], h[2]);
}
// h += A^T m  (A^T = A with a4, a5 negated)
__device__ __forceinline__ void mvT(float2 (&h)[3], const float (&a)[6], const float2 (&m)[3]) {
    h[0] = caxpy(a[0], m[0], h[0]); h[1] = caxpy(a[3], m[0], h[1]); h[2] = caxpy(a[4], m[0], h[2]);
    h[0] = caxpy(a[3], m[1], h[0]); h[1] = caxpy(a[1], m[1], h[1]); h[2] = caxpy(a[5], m[1], h[2]);
    h[0] = caxpy(-a[4], m[2], h[0]); h[1] = caxpy(-a[5], m[2], h[1]); h[2] = caxpy(a[2], m[2], h[2]);
}

}  // namespace

template <int NWARP, int NS, int MINB>
__global__ void __launch_bounds__(32 * NWARP, MINB)
coupling_symv_kernel(const float* __restrict__ bank, float2* __restrict__ spec, const float* __restrict__ inv_dz,
                     int nz, int batch, long long n_tiles, long long ks) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const SymvGeom G = symv_geom(nz);
    const int W = G.W, LW = G.LW, EPW = G.EPW;
    const int TE = NWARP * EPW;                              // entries per CTA tile; 2 TE spectrum slots per row
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int s = lane & 1, g = lane >> 1;                   // mirror slot, strip-lane
    const int ent = g >> G.log2LW, w = g & (LW - 1);         // entry of the warp-unit, strip
    const bool act = w < W;
    const uint32_t smask = s ? 0x80000000u : 0u;             // odd slot = mirror wavevector 2ny - ky: xy, yz change sign

    constexpr uint32_t STAGE = kSymvStageBytes;               // bytes of a full stage (four couples)
    const uint32_t bars = smem_u32(smem_raw) + warp * (NS * 8);
    const uint32_t ring = smem_u32(smem_raw) + ((NWARP * NS * 8 + 127) & ~127) + warp * (NS * STAGE);
    const uint32_t tile = smem_u32(smem_raw) + ((NWARP * NS * 8 + 127) & ~127) + NWARP * NS * STAGE;
    const uint32_t lane_off = (uint32_t)g * 16;

    // ---- this lane's slots in the M^ / H^ tile: row (c nz + 4 w + r), 16-byte chunk el ^ swizzle(w), half s ----
    const int el = warp * EPW + ent;
    const int chunk = el ^ ((w * EPW) & (TE - 1));
    const uint32_t my_off = (uint32_t)chunk * 16 + (uint32_t)s * 8;
    const uint32_t row_bytes = (uint32_t)TE * 16;
    const uint32_t tile_bytes = (uint32_t)(3 * nz) * row_bytes;     // two tile buffers: the next item's M^ arrives while this one is worked on

    // ---- bank ring: producer state (uniform over the warp; lane 0 issues) ----
    // this CTA's tiles: blockIdx.x, blockIdx.x + gridDim.x, ...; every tile is streamed once per state of the batch.
    // The bookkeeping is kept to a pointer, two counters and one comparison per stage: it runs once per 144 FFMA2.
    const int my_tiles = (int)((n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x);
    const uint32_t unit_bytes = (uint32_t)G.NC * kSymvCoupleBytes;
    const int stages_per_unit = G.SPE;                        // NC = 1 (mod 4): the last stage is one couple
    const long long tile_skip = (long long)gridDim.x * NWARP * unit_bytes - unit_bytes;
    const char* p_ptr = reinterpret_cast<const char*>(bank) + ((long long)blockIdx.x * NWARP + warp) * unit_bytes;
    int p_tiles = my_tiles, p_rep = batch, p_left = stages_per_unit;
    uint32_t cg = 0;
    const uint64_t pol = evict_first_policy();
    // fetch the next stage of the stream into ring slot `slot`
    auto produce = [&](uint32_t slot) {
        if (p_tiles > 0) {
            const uint32_t bytes = p_left == 1 ? (uint32_t)kSymvCoupleBytes : STAGE;
            if (lane == 0) {
                mbar_expect_tx(bars + slot * 8, bytes);
                bulk_g2s(ring + slot * STAGE, p_ptr, bytes, bars + slot * 8, pol);
            }
            p_ptr += bytes;
            if (--p_left == 0) {
                p_left = stages_per_unit;
                if (--p_rep == 0) { p_rep = batch; --p_tiles; p_ptr += tile_skip; }
                else p_ptr -= unit_bytes;
            }
        }
    };
    // wait for the next stage of the stream; returns this lane's address in it
    auto acquire = [&]() -> uint32_t {
        const uint32_t slot = cg & (NS - 1);
        mbar_wait(bars + slot * 8, (cg / NS) & 1);
        return ring + slot * STAGE + lane_off;
    };
    // the warp is done with the stage: refill it
    auto release = [&]() {
        const uint32_t slot = cg & (NS - 1);
        ++cg;
        __syncwarp();
        produce(slot);
    };

    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NS; ++i) mbar_init(bars + i * 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NS; ++i) produce(i);                 // the bank does not depend on the previous kernel

    pdl_wait();                                              // M^ comes from the previous kernel (S2)

    const int np = 3 * nz;
    const int log2TE = 3 + 4 - G.log2LW;                     // TE = NWARP EPW = 8 * 16 / LW
    static_assert(NWARP == 8, "log2TE assumes 8 warps per CTA");
    const int chunks_per_tile = np << log2TE;
    const int n_items = my_tiles * batch;
    // M^ tile of item n into buffer buf: rows of 16 TE bytes, chunk index swizzled by the strip of the row's layer
    auto fetch = [&](int n, int buf) {
        const int it = n / batch, b = n - it * batch;
        const long long t = blockIdx.x + (long long)it * gridDim.x;
        const float2* sp = spec + (long long)b * np * ks + t * (2 * TE);
        const uint32_t dst = tile + buf * tile_bytes;
        for (int x = tid; x < chunks_per_tile; x += 32 * NWARP) {
            const int lp = x >> log2TE, ch = x & (TE - 1);
            const int layer = lp - (lp >= 2 * nz ? 2 * nz : (lp >= nz ? nz : 0));
            const int chs = ch ^ (((layer >> 2) * EPW) & (TE - 1));
            cp_async16(dst + (uint32_t)lp * row_bytes + (uint32_t)chs * 16, sp + (long long)lp * ks + ch * 2);
        }
    };
    if (n_items > 0) fetch(0, 0);
    for (int n = 0; n < n_items; ++n) {
        const int it = n / batch, b = n - it * batch;
        const long long t = blockIdx.x + (long long)it * gridDim.x;
        float2* sp = spec + (long long)b * np * ks + t * (2 * TE);
        cp_async_wait_all();
        __syncthreads();                                     // this item's M^ has landed; the other buffer's H^ has been copied out
        if (n + 1 < n_items) fetch(n + 1, (n + 1) & 1);      // a different k range of the in-place spectrum: no hazard with this item's H^
        const uint32_t tbuf = tile + (n & 1) * tile_bytes;
        const uint32_t my_slot = tbuf + my_off;

        float2 mp[4][3], hp[4][3];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int layer = 4 * w + r;
            const bool live = act && layer < nz;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                mp[r][c] = live ? lds<float2>(my_slot + (uint32_t)(c * nz + layer) * row_bytes) : make_float2(0.f, 0.f);
                hp[r][c] = make_float2(0.f, 0.f);
            }
            mp[r][1] = make_float2(fxor(mp[r][1].x, smask), fxor(mp[r][1].y, smask));      // D M^ on the mirror slot
        }

        // ---- full blocks T = 1 .. nfull: strip w against strip (w + T) mod W ----
        int wp = w, wm = w;
        for (int T = 1; T <= G.nfull; ++T) {
            wp = wp + 1 == W ? 0 : wp + 1;
            wm = wm == 0 ? W - 1 : wm - 1;
            const int src_m = act ? (lane & ~(2 * LW - 2)) | (wp << 1) : lane;     // owner of the block's source layers
            const int src_c = act ? (lane & ~(2 * LW - 2)) | (wm << 1) : lane;     // strip whose block targets my layers
#pragma unroll
            for (int c2 = 0; c2 < 2; ++c2) {                 // one stage = two columns of the block
                const uint32_t st = acquire();
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    const int cc = 2 * c2 + hh;
                    float2 mq[3], cq[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) { mq[c] = shfl2(mp[cc][c], src_m); cq[c] = make_float2(0.f, 0.f); }
                    Couple k0, k1;
                    k0.load(st + hh * 2 * kSymvCoupleBytes);
                    k1.load(st + hh * 2 * kSymvCoupleBytes + kSymvCoupleBytes);
                    float a[6];
                    k0.get<0>(a); mv(hp[0], a, mq); mvT(cq, a, mp[0]);
                    k0.get<1>(a); mv(hp[1], a, mq); mvT(cq, a, mp[1]);
                    k1.get<0>(a); mv(hp[2], a, mq); mvT(cq, a, mp[2]);
                    k1.get<1>(a); mv(hp[3], a, mq); mvT(cq, a, mp[3]);
                    if (hh == 1) release();
#pragma unroll
                    for (int c = 0; c < 3; ++c) hp[cc][c] = cadd(hp[cc][c], shfl2(cq[c], src_c));
                }
            }
        }

        // ---- half block (W even): strip w against strip w + W/2, the block split between the two ----
        if (G.half) {
            const int wo = w < W / 2 ? w + W / 2 : w - W / 2;
            const int src = act ? (lane & ~(2 * LW - 2)) | (wo << 1) : lane;
            const bool lower = w < W / 2;
            const uint32_t tmask = lower ? 0u : 0x80000000u;      // the (r, r) pairs are stored as (lower, upper)
            const uint32_t other = act ? (uint32_t)(ent * LW + wo) * 16 - lane_off : 0u;
            float2 mq[3], cq[3];
            float a[6];
            Couple k0, k1;
            uint32_t st = acquire();
            k0.load(st);                                     // (0,1) (0,2)
            k1.load(st + kSymvCoupleBytes);                  // (1,2) (0,3)
            // column 1
#pragma unroll
            for (int c = 0; c < 3; ++c) { mq[c] = shfl2(mp[1][c], src); cq[c] = make_float2(0.f, 0.f); }
            k0.get<0>(a); mv(hp[0], a, mq); mvT(cq, a, mp[0]);
#pragma unroll
            for (int c = 0; c < 3; ++c) hp[1][c] = cadd(hp[1][c], shfl2(cq[c], src));
            // column 2
#pragma unroll
            for (int c = 0; c < 3; ++c) { mq[c] = shfl2(mp[2][c], src); cq[c] = make_float2(0.f, 0.f); }
            k0.get<1>(a); mv(hp[0], a, mq); mvT(cq, a, mp[0]);
            k1.get<0>(a); mv(hp[1], a, mq); mvT(cq, a, mp[1]);
#pragma unroll
            for (int c = 0; c < 3; ++c) hp[2][c] = cadd(hp[2][c], shfl2(cq[c], src));
            // column 3
#pragma unroll
            for (int c = 0; c < 3; ++c) { mq[c] = shfl2(mp[3][c], src); cq[c] = make_float2(0.f, 0.f); }
            k1.get<1>(a); mv(hp[0], a, mq); mvT(cq, a, mp[0]);
            k0.load(st + 2 * kSymvCoupleBytes);              // (1,3) (2,3)
            k0.get<0>(a); mv(hp[1], a, mq); mvT(cq, a, mp[1]);
            k0.get<1>(a); mv(hp[2], a, mq); mvT(cq, a, mp[2]);
#pragma unroll
            for (int c = 0; c < 3; ++c) hp[3][c] = cadd(hp[3][c], shfl2(cq[c], src));
            // (r, r): rows 0, 1 in the lower strip's couple, rows 2, 3 in the upper strip's; each strip does its own
            // direction of the product (the upper one with the transpose)
            k0.load(st + 3 * kSymvCoupleBytes + (lower ? 0u : other));
            k1.load(st + 3 * kSymvCoupleBytes + (lower ? other : 0u));
#pragma unroll
            for (int c = 0; c < 3; ++c) mq[c] = shfl2(mp[0][c], src);
            k0.get<0>(a, tmask); mv(hp[0], a, mq);
#pragma unroll
            for (int c = 0; c < 3; ++c) mq[c] = shfl2(mp[1][c], src);
            k0.get<1>(a, tmask); mv(hp[1], a, mq);
#pragma unroll
            for (int c = 0; c < 3; ++c) mq[c] = shfl2(mp[2][c], src);
            k1.get<0>(a, tmask); mv(hp[2], a, mq);
#pragma unroll
            for (int c = 0; c < 3; ++c) mq[c] = shfl2(mp[3][c], src);
            k1.get<1>(a, tmask); mv(hp[3], a, mq);
            release();
        }

        // ---- T = 0: inside the strip ----
        {
            float a[6];
            Couple k0, k1;
            uint32_t st = acquire();
            k0.load(st);                                     // (0,0) (1,1)
            k1.load(st + kSymvCoupleBytes);                  // (2,2) (3,3)
            k0.get<0>(a); mv(hp[0], a, mp[0]);
            k0.get<1>(a); mv(hp[1], a, mp[1]);
            k1.get<0>(a); mv(hp[2], a, mp[2]);
            k1.get<1>(a); mv(hp[3], a, mp[3]);
            k0.load(st + 2 * kSymvCoupleBytes);              // (0,1) (0,2)
            k1.load(st + 3 * kSymvCoupleBytes);              // (0,3) (1,2)
            k0.get<0>(a); mv(hp[0], a, mp[1]); mvT(hp[1], a, mp[0]);
            k0.get<1>(a); mv(hp[0], a, mp[2]); mvT(hp[2], a, mp[0]);
            k1.get<0>(a); mv(hp[0], a, mp[3]); mvT(hp[3], a, mp[0]);
            k1.get<1>(a); mv(hp[1], a, mp[2]); mvT(hp[2], a, mp[1]);
            release();
            st = acquire();
            k0.load(st);                                     // (1,3) (2,3)   (short stage: one couple)
            k0.get<0>(a); mv(hp[1], a, mp[3]); mvT(hp[3], a, mp[1]);
            k0.get<1>(a); mv(hp[2], a, mp[3]); mvT(hp[3], a, mp[2]);
            release();
        }

        // ---- H_i = (1 / dz_i) sum: back through the tile (each lane overwrites the slots it read) ----
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int layer = 4 * w + r;
            if (act && layer < nz) {
                const float sc = __ldg(inv_dz + layer);
#pragma unroll
                for (int c = 0; c < 3; ++c)                  // c == 1 on the mirror slot: back from D H^
                    sts(my_slot + (uint32_t)(c * nz + layer) * row_bytes, cscale(c == 1 ? fxor(sc, smask) : sc, hp[r][c]));
            }
        }
        __syncthreads();
        for (int x = tid; x < chunks_per_tile; x += 32 * NWARP) {
            const int lp = x >> log2TE, ch = x & (TE - 1);
            const int layer = lp - (lp >= 2 * nz ? 2 * nz : (lp >= nz ? nz : 0));
            const int chs = ch ^ (((layer >> 2) * EPW) & (TE - 1));
            const float4 v = lds128(tbuf + (uint32_t)lp * row_bytes + (uint32_t)chs * 16);
            *reinterpret_cast<float4*>(sp + (long long)lp * ks + ch * 2) = v;
        }
    }
}

bool coupling_symv_applies(int nz, size_t elem) { return elem == 4 && nz >= 2 && nz <= kSymvMaxNz; }

int coupling_symv_tile_entries(int nz) { return kSymvWarps * symv_geom(nz).EPW; }

size_t coupling_symv_bank_bytes(int nz, long long n_tiles) {
    const SymvGeom G = symv_geom(nz);
    return (size_t)n_tiles * kSymvWarps * G.NC * kSymvCoupleBytes;
}

cudaError_t launch_coupling_symv(const CouplingArgs& a, cudaStream_t st) {
    constexpr int NWARP = kSymvWarps, NS = 2, MINB = 2;       // ring: two stages of four couples per warp
    const SymvGeom G = symv_geom(a.nz);
    if (a.tile_k != 2 * NWARP * G.EPW) return cudaErrorInvalidValue;
    auto kern = coupling_symv_kernel<NWARP, NS, MINB>;
    const size_t smem = ((NWARP * NS * 8 + 127) & ~127) + (size_t)NWARP * NS * kSymvStageBytes +
                        (size_t)2 * 3 * a.nz * NWARP * G.EPW * 16;
    static PerDevice<int> cache;
    int occ = 1;
    cudaError_t err = ctas_per_sm_cached(kern, 32 * NWARP, smem, cache, occ);
    if (err != cudaSuccess) return err;
    long long grid = (long long)a.num_sms * occ;              // persistent CTAs; each walks its tiles for every state
    if (grid > a.n_tiles) grid = a.n_tiles;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(32 * NWARP), smem, st, (const float*)a.bank, (float2*)a.spec,
                      (const float*)a.inv_dz, a.nz, a.batch, a.n_tiles, a.ks);
}

}  // namespace hfft
