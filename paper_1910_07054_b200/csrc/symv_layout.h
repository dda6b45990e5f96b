// symv_layout.h -- layout of the reciprocity ("symmetric matvec") tensor bank read by coupling_symv.cu and written by
// tensor_build.cu (pack_symv_kernel); hfft_api.cu (hfft_read_bank) reads it back.  Host and device.
//
// Reciprocity (Eq.3 PAPER.md:38 is symmetric under the exchange of the two cuboids): with the real form R6 of
// the coupling and S_pq := dz_p R_pq one has S_qp = S_pq^T, so ONE stored 3 x 3 block serves two products,
//     H_p += S_pq M_q     and     H_q += S_pq^T M_p          (S^T = S with the xz, yz entries negated),
// and H_i = (1 / dz_i) (sum over q) at the end.  On top of the ky-mirror storage (one bank entry e = kx (ny+1) + t per
// wavevector pair ky = t, 2ny - t) the bank then holds nz (nz + 1) / 2 blocks per entry: a quarter of the plain bank.
//
// Schedule.  The nz layers are cut into W = ceil(nz / 4) strips of 4 rows; a strip is owned by a pair of lanes (one per
// mirror slot), 16 strip-lanes per warp, so a warp works on EPW = 16 / LW entries at a time (LW = W rounded up to a power
// of two).  The unordered strip pairs are visited round-robin: strip w meets strip (w + T) mod W at step T,
//     T = 1 .. nfull = (W - 1) / 2      full 4 x 4 blocks, 16 stored pairs per strip-lane (orientation p in w, q in w + T)
//     T = W / 2 (W even)                each of the two strips stores half of the block: the 6 pairs (r < c) in its own
//                                       orientation, and 2 of the 4 pairs (r, r) in the orientation (lower strip, upper)
//     T = 0                             inside the strip: 4 self pairs (r, r) and the 6 pairs (r < c)
// which is every unordered pair exactly once, the same number per strip-lane.  The stream of a warp-unit (EPW entries) is
// a sequence of NC "couples"; a couple holds two pairs (12 floats) for each of the 16 strip-lanes:
//     [unit][couple][j = 0..2][strip-lane g = 0..15][4 floats]          768 bytes per couple,
// float f = 6 h + c of a strip-lane (pair h = 0, 1 of the couple, component c = xx, yy, zz, xy, xz, yz) sits at j = f / 4,
// element f % 4.  Order of the couples: the full blocks T = 1 .. nfull (column cc = 0..3 of the block: couple 2 cc holds
// rows 0, 1, couple 2 cc + 1 rows 2, 3), then the half block (4 couples), then T = 0 (5 couples) -- so that every stage
// of four couples (3 KB) the kernel fetches ends on a block boundary and only the last stage of a unit is short (NC = 1 mod 4).
#pragma once

namespace hfft {

struct SymvGeom {
    int nz, W, LW, log2LW, EPW, nfull, half;
    int NC;      // couples per unit
    int SPE;     // stages (four couples; the last one a single couple) per unit
};

constexpr int kSymvCoupleFloats = 192;          // 16 strip-lanes x 12 floats
constexpr int kSymvCoupleBytes = 768;
constexpr int kSymvStageBytes = 4 * kSymvCoupleBytes;
constexpr int kSymvMaxNz = 64;                  // 16 strips of 4 rows

__host__ __device__ inline SymvGeom symv_geom(int nz) {
    SymvGeom g;
    g.nz = nz;
    g.W = (nz + 3) / 4;
    g.log2LW = 0;
    while ((1 << g.log2LW) < g.W) ++g.log2LW;
    g.LW = 1 << g.log2LW;
    g.EPW = g.LW <= 16 ? 16 / g.LW : 0;
    g.nfull = (g.W - 1) / 2;
    g.half = (g.W >= 2 && g.W % 2 == 0) ? 1 : 0;
    g.NC = 8 * g.nfull + 4 * g.half + 5;
    g.SPE = 2 * g.nfull + g.half + 2;
    return g;
}

// stored layer pairs per bank entry, padding included (what the stream costs; nz (nz + 1) / 2 without padding)
__host__ __device__ inline long long symv_pairs_per_entry(const SymvGeom& g) { return (long long)g.NC * 32 / g.EPW; }

// Where the block of the ordered pair (target i, source j) lives.  Returns the float offset, inside the unit's stream, of
// component 0 of the pair for entry-in-unit 0 -- add ent * LW * 4 floats for entry ent of the unit, and c (through
// symv_float_offset) for the component -- and sets transposed = 1 when the bank holds the orientation (j, i), i.e.
// S_ji = dz_j R_ji, from which S_ij = S_ji^T.
struct SymvPos { int couple, h, strip, transposed; };

__host__ __device__ inline SymvPos symv_pos(const SymvGeom& g, int i, int j) {
    // index of the pair (r, c), r <= c, inside a strip: self pairs first, then (r < c) -- order used by the T = 0 block
    const int wi = i >> 2, ri = i & 3, wj = j >> 2, rj = j & 3;
    SymvPos p;
    const int base_half = 8 * g.nfull, base_t0 = 8 * g.nfull + 4 * g.half;
    if (wi == wj) {
        const int r = ri < rj ? ri : rj, c = ri < rj ? rj : ri;
        // (0,0) (1,1) (2,2) (3,3) (0,1) (0,2) (0,3) (1,2) (1,3) (2,3)
        int idx;
        if (r == c) idx = r;
        else idx = 4 + (r == 0 ? c - 1 : (r == 1 ? c + 1 : 5));
        p.couple = base_t0 + idx / 2; p.h = idx & 1; p.strip = wi; p.transposed = ri > rj;
        return p;
    }
    int d = wj - wi;
    if (d < 0) d += g.W;                                    // strip wj = wi + d (mod W)
    if (d >= 1 && d <= g.nfull) {                           // stored by strip wi as (row ri, column rj of the block T = d)
        p.couple = (d - 1) * 8 + 2 * rj + (ri >> 1); p.h = ri & 1; p.strip = wi; p.transposed = 0;
        return p;
    }
    if (g.W - d >= 1 && g.W - d <= g.nfull) {               // stored by strip wj as (row rj, column ri of the block T = W - d)
        p.couple = (g.W - d - 1) * 8 + 2 * ri + (rj >> 1); p.h = rj & 1; p.strip = wj; p.transposed = 1;
        return p;
    }
    // half block: d == W / 2
    if (ri != rj) {
        // pairs (r < c) in the order (0,1) (0,2) (1,2) (0,3) (1,3) (2,3), stored by the strip that owns row r
        const bool own = ri < rj;
        const int r = own ? ri : rj, c = own ? rj : ri;
        const int idx = c == 1 ? 0 : (c == 2 ? 1 + r : 3 + r);
        p.couple = base_half + idx / 2; p.h = idx & 1; p.strip = own ? wi : wj; p.transposed = own ? 0 : 1;
        return p;
    }
    // (r, r): orientation (lower strip, upper strip); rows 0, 1 in the lower strip's couple, rows 2, 3 in the upper one's
    const int lo = wi < wj ? wi : wj, hi = wi < wj ? wj : wi;
    p.couple = base_half + 3; p.h = ri & 1; p.strip = ri < 2 ? lo : hi; p.transposed = wi == lo ? 0 : 1;
    return p;
}

// float offset inside the unit's stream of component c of a pair at position p, for entry-in-unit ent
__host__ __device__ inline long long symv_float_offset(const SymvGeom& g, const SymvPos& p, int ent, int c) {
    const int f = 6 * p.h + c, gl = ent * g.LW + p.strip;
    return (long long)p.couple * kSymvCoupleFloats + (f >> 2) * 64 + gl * 4 + (f & 3);
}

}  // namespace hfft
