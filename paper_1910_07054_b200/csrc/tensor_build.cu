// tensor_build.cu -- stage S0 (timed setup): the spectral tensor bank F1F2(N_kl)_{i3-j3} of Eq.24
// (PAPER.md:177-178), built on the device.
//
// Tensor (PAPER.md:52 Eq.5, :99 Eq.11 with the 4th term read as Y+dy [A1], :249-291 Eq.27-31).
// Multiplying out Eq.5 x Eq.28 x Eq.27 (F2 -> f) and Eq.11 x Eq.31 x Eq.30
// (G2 -> g) gives, for all six components c with their permuted primitive phi_c
// (newell_dd.cuh), one signed 4 x 4 x 4 stencil.  In the plane target and source cells have the
// same size, so the x and y stencils collapse to second differences; along z the four points are
// the interface differences of the two layers (Z_ij = zeta_i - zeta_j, lower faces, reading A8):
//
//   Psi_c(a, b)(p, q) = sum_{al,be in {-1,0,1}} w_al w_be phi_c((p+al) dx, (q+be) dy, zeta_a - zeta_b),
//                       w = (1, -2, 1)
//   N^c_ij(p dx, q dy) = -1 / (4 pi dx dy dz_i) [ Psi_c(i+1, j) - Psi_c(i, j) - Psi_c(i+1, j+1) + Psi_c(i, j+1) ]
//
// with |tau| = dx dy dz_i the TARGET volume (reading A7).  Everything up to the
// rounding of N to fp64 runs in double-double (reading A16).
//
// Then: N is laid on the 2nx x 2ny periodic grid at (p mod 2nx, q mod 2ny), the slots p = nx and
// q = ny are 0 (reading A10), negative offsets come from the parities of the components (xx, yy,
// zz even in X and Y; xy odd, odd; xz odd, even; yz even, odd); a full (not zero-padded) fp64
// real-to-complex 2-D FFT follows, and the real part (xx, yy, zz, xy) or imaginary part (xz, yz)
// times -1/(4 nx ny) is stored in the plan precision at bank[tile][i][j][c][k in tile].
#include <math.h>

#include <map>
#include <utility>

#include "hfft_internal.h"
#include "newell_dd.cuh"
#include "symv_layout.h"

namespace hfft {

__constant__ int kParX[6] = {+1, +1, +1, -1, -1, +1};
__constant__ int kParY[6] = {+1, +1, +1, -1, +1, -1};
__constant__ int kParZ[6] = {+1, +1, +1, +1, -1, -1};

// phi[b][c][Q][P], Q in [0, ny], P in [0, nx], z = zeta[a] - zeta[b]
__global__ void __launch_bounds__(128)
lattice_kernel(double2* __restrict__ phi, const double2* __restrict__ zeta, int a, int b0, int nx, int ny, int nz,
               double dx, double dy) {
    const int P = blockIdx.x * blockDim.x + threadIdx.x;
    const int Q = blockIdx.y;
    const int b = b0 + blockIdx.z;
    if (P > nx) return;
    dd za = dd_make(zeta[a].x, zeta[a].y), zb = dd_make(zeta[b].x, zeta[b].y);
    dd z = dd_sub(za, zb);
    const bool zneg = z.hi < 0.0;
    z = dd_abs(z);
    dd x = two_prod((double)P, dx), y = two_prod((double)Q, dy);
    dd v[6];
    newell_phi6(x, y, z, v);
    const size_t plane = (size_t)(ny + 1) * (nx + 1);
    size_t o = (size_t)b * 6 * plane + (size_t)Q * (nx + 1) + P;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        dd u = (zneg && kParZ[c] < 0) ? dd_neg(v[c]) : v[c];
        phi[o + c * plane] = make_double2(u.hi, u.lo);
    }
}

// psi[b][c][q][p] = second difference in x and in y of phi, p in [0, nx), q in [0, ny)
__global__ void __launch_bounds__(128)
stencil_kernel(double2* __restrict__ psi, const double2* __restrict__ phi, int bc0, int nx, int ny) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int q = blockIdx.y;
    const int bc = bc0 + blockIdx.z;    // b * 6 + c
    if (p >= nx) return;
    const int c = bc % 6;
    const double2* f = phi + (size_t)bc * (ny + 1) * (nx + 1);
    dd acc = dd_make(0.0, 0.0);
#pragma unroll
    for (int be = -1; be <= 1; ++be) {
        int Q = q + be;
        double sy = 1.0;
        if (Q < 0) { Q = -Q; sy = (double)kParY[c]; }
        dd row = dd_make(0.0, 0.0);
#pragma unroll
        for (int al = -1; al <= 1; ++al) {
            int P = p + al;
            double sx = 1.0;
            if (P < 0) { P = -P; sx = (double)kParX[c]; }
            double2 t = f[(size_t)Q * (nx + 1) + P];
            double w = (al == 0 ? -2.0 : 1.0) * sx;
            row = dd_add(row, dd_make(t.x * w, t.y * w));
        }
        double w = (be == 0 ? -2.0 : 1.0) * sy;
        acc = dd_add(acc, dd_make(row.hi * w, row.lo * w));
    }
    psi[((size_t)bc * ny + q) * nx + p] = make_double2(acc.hi, acc.lo);
}

// N^c_ij on the padded periodic grid: R[jl][c][2ny][2nx] (fp64), jl = j - j0
__global__ void __launch_bounds__(128)
assemble_kernel(double* __restrict__ R, const double2* __restrict__ psi_lo /* a = i */,
                const double2* __restrict__ psi_hi /* a = i+1 */, int nx, int ny, int j0, double2 neg_inv_4pi_tau) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int q = blockIdx.y;
    const int jc = blockIdx.z;          // jl * 6 + c
    if (p >= nx) return;
    const int jl = jc / 6, c = jc - jl * 6;
    const int j = j0 + jl;
    const size_t pl = (size_t)ny * nx;
    const size_t o = (size_t)q * nx + p;
    auto ld = [&](const double2* s, int b) {
        double2 t = s[((size_t)b * 6 + c) * pl + o];
        return dd_make(t.x, t.y);
    };
    dd s = dd_sub(ld(psi_hi, j), ld(psi_lo, j));
    s = dd_sub(s, ld(psi_hi, j + 1));
    s = dd_add(s, ld(psi_lo, j + 1));
    s = dd_mul(s, dd_make(neg_inv_4pi_tau.x, neg_inv_4pi_tau.y));
    const double v = s.hi;
    const double sx = (double)kParX[c], sy = (double)kParY[c];
    double* dst = R + (size_t)jc * 4 * pl;
    const int W = 2 * nx, H = 2 * ny;
    dst[(size_t)q * W + p] = v;
    if (p > 0) dst[(size_t)q * W + (W - p)] = v * sx;
    if (q > 0) dst[(size_t)(H - q) * W + p] = v * sy;
    if (p > 0 && q > 0) dst[(size_t)(H - q) * W + (W - p)] = v * sx * sy;
}

// bank entry e of a (pair, component): tile_e entries per tile, n_e entries (padded to whole tiles: n_e_padded).
// Plain layout: e = k.  Mirror layout (fft_kernels.cu ypos): e = kx * (ny + 1) + t, t = 0..ny, taken from k = kx * 2ny + t.
template <typename T>
__global__ void __launch_bounds__(256)
pack_kernel(T* __restrict__ bank, const double2* __restrict__ Y, int nz, int i, int j0, int ncls,
            const unsigned short* __restrict__ cls, int tile_e, long long n_k, long long n_e, long long n_e_padded,
            int mirror_ny, double scale) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int jc = blockIdx.y;          // jl * 6 + c
    if (e >= n_e_padded) return;
    const int jl = jc / 6, c = jc - jl * 6;
    double v = 0.0;
    if (e < n_e) {
        long long k = e;
        if (mirror_ny > 0) {
            const long long kx = e / (mirror_ny + 1);
            k = kx * 2 * mirror_ny + (e - kx * (mirror_ny + 1));
        }
        double2 t = Y[(size_t)jc * n_k + k];
        v = (c < 4 ? t.x : t.y) * scale;
    }
    const long long tile = e / tile_e;
    const int kk = (int)(e - tile * tile_e);
    const int pr = i * nz + j0 + jl;                       // bank slot = tensor class of the pair
    const long long blk = (tile * ncls + (cls ? (int)cls[pr] : pr)) * 6LL * tile_e;
    if (mirror_ny > 0) {
        // [component pair][lane][2][KB]: a lane's two components of a pair are one 16-byte vector (coupling.cu MIR)
        const int KB = tile_e / 32, lane = kk / KB, kl = kk - lane * KB;
        bank[blk + (((c >> 1) * 32 + lane) * 2 + (c & 1)) * KB + kl] = (T)v;
    } else {
        bank[blk + (long long)c * tile_e + kk] = (T)v;
    }
}

// Reciprocity bank in the symv layout (symv_layout.h): the pairs (i, j0 + jl) of a run are stored orientations, their
// value S_ij = dz_i R_ij (the factor is in `scale`) goes to [unit = e / EPW][couple][...] for bank entry e = kx (ny + 1) + t.
__global__ void __launch_bounds__(256)
pack_symv_kernel(float* __restrict__ bank, const double2* __restrict__ Y, int nz, int i, int j0, long long n_k, long long n_e,
                 int ny, double scale) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int jc = blockIdx.y;          // jl * 6 + c
    if (e >= n_e) return;               // padding entries and padding rows stay zero (the bank is cleared first)
    const int jl = jc / 6, c = jc - jl * 6;
    const SymvGeom G = symv_geom(nz);
    const SymvPos pos = symv_pos(G, i, j0 + jl);
    const long long kx = e / (ny + 1);
    const long long k = kx * 2 * ny + (e - kx * (ny + 1));
    const double2 t = Y[(size_t)jc * n_k + k];
    const double v = (c < 4 ? t.x : t.y) * scale;
    const long long unit = e / G.EPW;
    const int ent = (int)(e - unit * G.EPW);
    bank[unit * G.NC * kSymvCoupleFloats + symv_float_offset(G, pos, ent, c)] = (float)v;
}

struct ScratchLayout {
    size_t zeta, cls, phi, psi0, psi1, R, X, Y, total;
    int jc;
};

static ScratchLayout scratch_layout(const BuildGeom& g) {
    ScratchLayout L;
    auto al = [](size_t v) { return (v + 255) & ~(size_t)255; };
    const size_t nxy = (size_t)g.nx * g.ny;
    const size_t per_j = 6 * (4 * nxy * 8 + 2 * (size_t)g.n_k * 16);
    size_t jc = ((size_t)1 << 30) / per_j;
    if (jc < 1) jc = 1;
    if (jc > (size_t)g.nz) jc = g.nz;
    L.jc = (int)jc;
    size_t o = 0;
    L.zeta = o; o += al((size_t)(g.nz + 1) * 16);
    L.cls = o;  o += al((size_t)g.nz * g.nz * sizeof(unsigned short));
    L.phi = o;  o += al((size_t)(g.nz + 1) * 6 * (g.ny + 1) * (g.nx + 1) * 16);
    L.psi0 = o; o += al((size_t)(g.nz + 1) * 6 * nxy * 16);
    L.psi1 = o; o += al((size_t)(g.nz + 1) * 6 * nxy * 16);
    L.R = o;    o += al(jc * 6 * 4 * nxy * 8);
    L.X = o;    o += al(jc * 6 * (size_t)g.n_k * 16);
    L.Y = o;    o += al(jc * 6 * (size_t)g.n_k * 16);
    L.total = o;
    return L;
}

size_t build_scratch_bytes(const BuildGeom& g) { return scratch_layout(g).total; }

#define HFFT_CK(call)                                                                  \
    do {                                                                               \
        cudaError_t e_ = (call);                                                       \
        if (e_ != cudaSuccess) {                                                       \
            err = std::string(#call) + ": " + cudaGetErrorString(e_);                  \
            return e_;                                                                 \
        }                                                                              \
    } while (0)

// Source layers j of target row i whose tensor has to be evaluated, as inclusive runs [j0, j1].
//  - hfft_update_dz (changed >= 0): N_ij depends on (dz_i, dz_j, zeta_i - zeta_j) only, so pairs
//    on one side of the changed layer keep their tensor;
//  - deduplicated bank (g.pair_class): only the representative pair of every tensor class;
//  - reciprocity storage (g.pair_class = slot of the unordered pair): the stored orientation of every pair, and with
//    changed >= 0 only the pairs that straddle or contain the changed layer.
static std::vector<std::pair<int, int>> row_runs(const BuildGeom& g, int changed, int i) {
    const int nz = g.nz;
    std::vector<std::pair<int, int>> runs;
    if (!g.pair_class) {
        int jlo = 0, jhi = nz - 1;
        if (changed >= 0 && i != changed) { if (i < changed) jlo = changed; else jhi = changed; }
        runs.push_back({jlo, jhi});
        return runs;
    }
    for (int j = 0; j < nz; ++j) {
        if (g.class_rep[g.pair_class[i * nz + j]] != i * nz + j) continue;
        // reciprocity storage + hfft_update_dz: of the stored orientations only those whose pair has the changed layer
        // between (or at) its two layers get a new tensor; S_pq = dz_p R_pq changes with dz_p only for p == changed,
        // which is one of them
        if (changed >= 0 && !((i <= changed && changed <= j) || (j <= changed && changed <= i))) continue;
        if (!runs.empty() && runs.back().second == j - 1) runs.back().second = j;
        else runs.push_back({j, j});
    }
    return runs;
}

// Tensor classes: N_ij is a function of (dz_i, dz_j, Z_ij = zeta_i - zeta_j) alone (PAPER.md:150
// Eq.19 with Eq.5/11), so pairs that agree in all three share one bank slot.  dz must agree bit for bit, Z (a
// double-double difference of the interface coordinates) to 2^-80 of the stack height.  If the class depends on
// i - j only (equal thicknesses: the z-convolution of Eq.24 is a Toeplitz one, the case of the paper's equidistant
// comparison) the classes are folded to |i - j| (see below).
void pair_classes(int nz, const double* dz, std::vector<int>& cls, std::vector<int>& rep, bool& toeplitz) {
    std::vector<dd> zeta(nz + 1);
    zeta[0] = dd_make(0.0, 0.0);
    for (int k = 0; k < nz; ++k) zeta[k + 1] = dd_add_d(zeta[k], dz[k]);
    const double tol = ldexp(zeta[nz].hi, -80);
    struct Key {
        double a, b, z;
        bool operator<(const Key& o) const { return a != o.a ? a < o.a : (b != o.b ? b < o.b : z < o.z); }
    };
    std::map<Key, std::vector<int>> seen;        // key -> classes with that (dz_i, dz_j, Z.hi)
    std::vector<dd> zcls;
    cls.assign((size_t)nz * nz, 0);
    rep.clear();
    for (int i = 0; i < nz; ++i)
        for (int j = 0; j < nz; ++j) {
            const dd Z = dd_sub(zeta[i], zeta[j]);
            std::vector<int>& cand = seen[Key{dz[i], dz[j], Z.hi}];
            int c = -1;
            for (int t : cand) {
                const dd d = dd_sub(Z, zcls[t]);
                if (fabs(d.hi) <= tol) { c = t; break; }
            }
            if (c < 0) { c = (int)rep.size(); rep.push_back(i * nz + j); zcls.push_back(Z); cand.push_back(c); }
            cls[(size_t)i * nz + j] = c;
        }
    toeplitz = nz > 1;
    for (int i = 0; i + 1 < nz && toeplitz; ++i)
        for (int j = 0; j + 1 < nz; ++j)
            if (cls[(size_t)i * nz + j] != cls[(size_t)(i + 1) * nz + j + 1]) { toeplitz = false; break; }
    if (toeplitz && (int)rep.size() == 2 * nz - 1) {
        // equal thicknesses: N_ij depends on d = i - j only, and N_{-d} = N_d except that xz and yz change sign
        // (reciprocity dz_i N_ij(X,Y) = dz_j N_ji(-X,-Y) with the in-plane parities of the components: xx, yy, zz,
        // xy are even under (X,Y) -> (-X,-Y), xz and yz odd).  One slot per |d|, representative pair (d, 0); the
        // kernels negate the xz, yz entries for i < j.
        rep.assign(nz, 0);
        for (int i = 0; i < nz; ++i)
            for (int j = 0; j < nz; ++j) cls[(size_t)i * nz + j] = i >= j ? i - j : j - i;
        for (int d = 0; d < nz; ++d) rep[d] = d * nz;
    } else {
        toeplitz = false;
    }
}

cudaError_t build_bank(const BuildGeom& g, void* bank, void* scratch, const void* tw2nx, const void* twt_nx,
                       const void* twt_2ny, int changed, cudaStream_t st, std::string& err) {
    const ScratchLayout L = scratch_layout(g);
    unsigned char* base = static_cast<unsigned char*>(scratch);
    double2* d_zeta = reinterpret_cast<double2*>(base + L.zeta);
    double2* d_phi = reinterpret_cast<double2*>(base + L.phi);
    double2* d_psi[2] = {reinterpret_cast<double2*>(base + L.psi0), reinterpret_cast<double2*>(base + L.psi1)};
    double* d_R = reinterpret_cast<double*>(base + L.R);
    double2* d_X = reinterpret_cast<double2*>(base + L.X);
    double2* d_Y = reinterpret_cast<double2*>(base + L.Y);
    const int nx = g.nx, ny = g.ny, nz = g.nz;

    // lower-face coordinates zeta_0 = 0, zeta_{k+1} = zeta_k + dz_k in double-double (reading A8/A9)
    std::vector<double2> zeta(nz + 1);
    dd acc = dd_make(0.0, 0.0);
    zeta[0] = make_double2(0.0, 0.0);
    for (int k = 0; k < nz; ++k) {
        acc = dd_add_d(acc, g.dz[k]);
        zeta[k + 1] = make_double2(acc.hi, acc.lo);
    }
    HFFT_CK(cudaMemcpyAsync(d_zeta, zeta.data(), sizeof(double2) * (nz + 1), cudaMemcpyHostToDevice, st));
    unsigned short* d_cls = nullptr;
    std::vector<unsigned short> cls16;
    if (g.pair_class) {
        d_cls = reinterpret_cast<unsigned short*>(base + L.cls);
        cls16.assign(g.pair_class, g.pair_class + (size_t)nz * nz);
        HFFT_CK(cudaMemcpyAsync(d_cls, cls16.data(), cls16.size() * sizeof(unsigned short), cudaMemcpyHostToDevice, st));
    }
    const int ncls = g.pair_class ? g.n_classes : nz * nz;
    HFFT_CK(cudaStreamSynchronize(st));   // `zeta`, `cls16` are pageable host memory
    HFFT_CK(cudaMemsetAsync(d_R, 0, (size_t)L.jc * 6 * 4 * nx * ny * 8, st));   // slots p = nx, q = ny stay 0
    // symv layout: padding rows (nz not a multiple of 4), idle strip-lanes and padding entries hold zeros
    if (g.symv && changed < 0) HFFT_CK(cudaMemsetAsync(bank, 0, g.symv_bank_bytes, st));

    const double scale = -1.0 / (4.0 * (double)nx * (double)ny);
    const dd inv4pi = dd_make(DD_INV_4PI_HI, DD_INV_4PI_LO);
    std::vector<std::vector<std::pair<int, int>>> runs(nz);
    for (int i = 0; i < nz; ++i) runs[i] = row_runs(g, changed, i);
    for (int a = 0; a <= nz; ++a) {
        {
            // interface a serves target rows a - 1 (upper face) and a (lower face): source interfaces b
            // in the union of their ranges [jlo, jhi + 1]
            int blo = nz + 1, bhi = -1;
            for (int i = a - 1; i <= a; ++i) {
                if (i < 0 || i >= nz || runs[i].empty()) continue;
                if (runs[i].front().first < blo) blo = runs[i].front().first;
                if (runs[i].back().second + 1 > bhi) bhi = runs[i].back().second + 1;
            }
            if (bhi >= blo) {
                dim3 grid((nx + 1 + 127) / 128, ny + 1, bhi - blo + 1);
                lattice_kernel<<<grid, 128, 0, st>>>(d_phi, d_zeta, a, blo, nx, ny, nz, g.dx, g.dy);
                HFFT_CK(cudaGetLastError());
                dim3 grid2((nx + 127) / 128, ny, (bhi - blo + 1) * 6);
                stencil_kernel<<<grid2, 128, 0, st>>>(d_psi[a & 1], d_phi, blo * 6, nx, ny);
                HFFT_CK(cudaGetLastError());
            }
        }
        if (a == 0) continue;
        const int i = a - 1;
        // -1 / (4 pi dx dy dz_i) in double-double
        dd tau = dd_mul_d(two_prod(g.dx, g.dy), g.dz[i]);
        dd coef = dd_neg(dd_div(inv4pi, tau));
        // reciprocity storage keeps S_ij = dz_i R_ij (then S_ji = S_ij^T): the factor goes into the packing
        const double pscale = g.recip ? scale * g.dz[i] : scale;
        for (const auto& run : runs[i])
            for (int j0 = run.first; j0 <= run.second; j0 += L.jc) {
                const int jn = (run.second + 1 - j0 < L.jc) ? run.second + 1 - j0 : L.jc;
                dim3 grid((nx + 127) / 128, ny, jn * 6);
                assemble_kernel<<<grid, 128, 0, st>>>(d_R, d_psi[i & 1], d_psi[a & 1], nx, ny, j0,
                                                      make_double2(coef.hi, coef.lo));
                HFFT_CK(cudaGetLastError());
                HFFT_CK((launch_fftx_fwd<double, false>(d_R, d_X, g.log2nx, jn * 6, 2 * ny, 0, nullptr, tw2nx, twt_nx,
                                                        g.num_sms, st)));
                HFFT_CK((launch_ffty_fwd<double, false>(d_X, d_Y, nx, g.log2ny + 1, jn * 6, 0, g.n_k, twt_2ny,
                                                        g.num_sms, st)));
                const int tile_e = g.mirror ? g.tile_k / 2 : g.tile_k;
                const long long n_e = g.mirror ? (long long)(nx + 1) * (ny + 1) : g.n_k;
                const long long n_e_padded = g.mirror ? g.n_k_padded / 2 : g.n_k_padded;
                dim3 gridp((unsigned)((n_e_padded + 255) / 256), jn * 6);
                if (g.symv)
                    pack_symv_kernel<<<dim3((unsigned)((n_e + 255) / 256), jn * 6), 256, 0, st>>>((float*)bank, d_Y, nz, i, j0, g.n_k,
                                                                                              n_e, ny, pscale);
                else if (g.prec == HFFT_F32)
                    pack_kernel<float><<<gridp, 256, 0, st>>>((float*)bank, d_Y, nz, i, j0, ncls, d_cls, tile_e, g.n_k, n_e,
                                                              n_e_padded, g.mirror ? ny : 0, pscale);
                else
                    pack_kernel<double><<<gridp, 256, 0, st>>>((double*)bank, d_Y, nz, i, j0, ncls, d_cls, tile_e, g.n_k,
                                                               n_e, n_e_padded, g.mirror ? ny : 0, pscale);
                HFFT_CK(cudaGetLastError());
            }
    }
    HFFT_CK(cudaStreamSynchronize(st));
    return cudaSuccess;
}

}  // namespace hfft
