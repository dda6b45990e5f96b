// hfft_internal.h -- declarations shared by the translation units of libhfft (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdlib.h>
#include <map>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "../../include/hfft.h"

namespace hfft {

// Launch of a hot-path kernel with programmatic dependent launch (PDL): the kernel may start -- run its prologue:
// index arithmetic, twiddle registers, shared-memory addresses -- while the previous kernel of the stream drains;
// every such kernel executes pdl_wait() (fft.cuh: griddepcontrol.wait) before it touches data that kernel wrote.
// Takes the launch gaps out of the five-kernel evaluation (B200, C3: 0.147 -> see DESIGN.md 8).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    static const int pdl_on = getenv("HFFT_NO_PDL") ? 0 : 1;      // HFFT_NO_PDL=1: plain stream order (A/B measurements)
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = pdl_on;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// Launch attributes are properties of a (kernel, device) pair: the opt-in to more than 48 KB of dynamic shared memory
// (cudaFuncSetAttribute) and the occupancy the runtime reports.  Every launcher keeps them in one of these caches,
// keyed by device ordinal and a launcher-defined key (threads, shared-memory bytes), guarded by a mutex, so that
// plans on several devices or host threads of one process do not share stale values.
template <typename V> class PerDevice {
  public:
    bool get(int dev, long long key, V& out) {
        std::lock_guard<std::mutex> lock(mu_);
        return get_locked(dev, key, out);
    }
    void set(int dev, long long key, const V& v) {
        std::lock_guard<std::mutex> lock(mu_);
        map_[std::make_pair(dev, key)] = v;
    }
    // for read-modify-write sequences that must not interleave between host threads (ctas_per_sm_cached)
    std::mutex& mutex() { return mu_; }
    bool get_locked(int dev, long long key, V& out) const {
        auto it = map_.find(std::make_pair(dev, key));
        if (it == map_.end()) return false;
        out = it->second;
        return true;
    }
    void set_locked(int dev, long long key, const V& v) { map_[std::make_pair(dev, key)] = v; }
  private:
    std::mutex mu_;
    std::map<std::pair<int, long long>, V> map_;
};

// CTAs per SM of `kernel` launched with (threads, smem) on the current device, opting in to smem > 48 KB first.
// The opt-in is one attribute per (kernel, device) that every call overwrites: it is only ever raised (key -1 of the
// cache holds the value in force), so that a launch whose occupancy is cached never finds it lowered by a later,
// smaller configuration.  The look-up of the value in force, cudaFuncSetAttribute and the update of key -1 happen
// under ONE lock: two host threads that bring the same kernel up with different shared-memory sizes cannot leave the
// attribute at the smaller value while the cache records the larger one.
template <typename K>
inline cudaError_t ctas_per_sm_cached(K kernel, int threads, size_t smem, PerDevice<int>& cache, int& occ) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const long long key = ((long long)threads << 32) | (long long)smem;
    std::lock_guard<std::mutex> lock(cache.mutex());
    if (cache.get_locked(dev, key, occ)) return cudaSuccess;
    int opted = 48 * 1024;
    cache.get_locked(dev, -1, opted);
    if ((int)smem > opted) {
        if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess)
            return e;
        cache.set_locked(dev, -1, (int)smem);
    }
    int nb = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, threads, smem)) != cudaSuccess) return e;
    occ = nb < 1 ? 1 : nb;
    cache.set_locked(dev, key, occ);
    return cudaSuccess;
}

// per-layer saturation magnetisation, passed by value to the S1 kernel (hfft.h: "read during the
// call and passed by value to the kernels")
template <typename T> struct MsParam { T v[HFFT_MAX_NZ]; };

// ---- fft_kernels.cu ----
// tw2nx: exp(-2 pi i t / 2nx), 2nx entries (split / merge of the packed real transform);
// twt_*: per-thread twiddle table of the row transform (layout in fft.cuh; host: thread_twiddle_table)
// forward x: `in` real rows [nplanes][rows_per_plane][nx if ZP else 2nx] -> X^ [nplanes][nx+1][rows_per_plane]
template <typename T, bool ZP>
cudaError_t launch_fftx_fwd(const T* in, void* xhat, int log2nx, int nplanes, int rows_per_plane, int nz,
                            const double* ms_host, const void* tw2nx, const void* twt_nx, int num_sms,
                            cudaStream_t st);
// sums != nullptr: also accumulate sums[plane][2] += (sum of out, sum of m * out) over the plane's cells
template <typename T>
cudaError_t launch_ifftx(const void* xhat, T* out, int log2nx, int nplanes, int rows_per_plane, const void* tw2nx,
                         const void* twt_nx, int num_sms, const T* m, double* sums, cudaStream_t st);
// forward y: X^ rows [nplanes * (nx+1)][N/2 if ZP else N] -> k side [nplanes][ks], k = kx * N + ky
// (mirror: kx * (N + 2) + ypos(ky), ky and N - ky in adjacent slots; fft_kernels.cu);
// nz_rot > 0 multiplies the z-component planes by i
template <typename T, bool ZP>
cudaError_t launch_ffty_fwd(const void* xhat, void* spec, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                            const void* twt_N, int num_sms, cudaStream_t st, int mirror = 0);
template <typename T>
cudaError_t launch_iffty(const void* spec, void* xhat, int nx, int log2N, int nplanes, int nz_rot, long long ks,
                         const void* twt_N, int num_sms, cudaStream_t st, int mirror = 0);

// ---- fused_ycy.cu: S2 + S3 + S4 in one kernel, one kx column of all planes per CTA (plain bank, tile_k == 32) ----
size_t fused_ycy_smem_bytes(int log2N, int nz, size_t elem);   // 0: shape not supported
bool fused_ycy_pays(int log2N, int nz, size_t elem);           // automatic mode: the bank slice fits shared memory too
template <typename T>
cudaError_t launch_fused_ycy(void* xhat, const void* bank, int nx, int log2N, int nz, int batch, const void* twt_N, int num_sms,
                             cudaStream_t st);

// ---- coupling.cu ----
// H^ = bank * M^ in place on the k side.  bank layout [tile][class][6][tile_k]; class = i*nz+j (cls == nullptr)
// or cls[i*nz+j] (deduplicated bank, device table).
struct CouplingArgs {
    const void* bank; void* spec;
    int nz, batch, tile_k;
    long long n_tiles, ks;
    int n_classes;                 // nz*nz without deduplication
    const unsigned short* cls;     // device, [nz*nz], or nullptr
    bool class_kernel;             // bank tile in shared memory (coupling_class_applies)
    bool toeplitz;                 // equal thicknesses: cls[i*nz+j] == |i - j|, xz / yz negated for i < j
    int num_sms;
    // z-FFT mode (coupling_zfft.cu; Eq.25): bank = S(k, kz) [tile][kz][6][32], Lz = 2^log2lz
    bool recip = false;            // reciprocity storage: cls = slot of the unordered pair, bank = dz_p R_pq (p <= q)
    const void* inv_dz = nullptr;  // device, [nz] plan precision (recip)
    bool mirror = false;           // spectrum in the mirror layout, one bank value per pair of slots (coupling_kernel MIR)
    bool symv = false;             // reciprocity bank in the symv layout (coupling_symv.cu, symv_layout.h); fp32
    bool zfft = false;
    int log2lz = 0;
    const void* twz = nullptr;     // device, exp(-2 pi i n / Lz), plan precision
};
template <typename T>
cudaError_t launch_coupling(const CouplingArgs& a, cudaStream_t st);
// ---- coupling_symv.cu ----
constexpr int kSymvWarps = 8;      // warps per CTA of coupling_symv_kernel; a CTA tile is kSymvWarps * EPW bank entries
bool coupling_symv_applies(int nz, size_t elem);
int coupling_symv_tile_entries(int nz);
size_t coupling_symv_bank_bytes(int nz, long long n_tiles);
cudaError_t launch_coupling_symv(const CouplingArgs& a, cudaStream_t st);
// ---- coupling_zfft.cu ----
template <typename T>
cudaError_t launch_coupling_zfft(const CouplingArgs& a, cudaStream_t st);
bool coupling_zfft_applies(int nz, size_t elem, int* log2lz);
// bank3 [tile][kz][6][32] (plan precision) from the fp64 Toeplitz classes cls64 [nz][6][kstride]
cudaError_t launch_zdft_bank(void* bank3, const double* cls64, const void* twz64, int nz, int log2lz, long long n_k,
                             long long kstride, long long n_k_padded, int prec, cudaStream_t st);

// shared-memory-resident class kernel: needs tile_k == 32 and this many bytes per CTA
size_t coupling_class_smem_bytes(int nz, int n_classes, bool toeplitz, size_t elem);
size_t coupling_smem_bytes(int nz, int tile_k, size_t elem);
// batched register-resident-bank kernel (B > 1, small nz); it needs tile_k == 32
bool coupling_batched_applies(int nz, int batch, size_t elem);

// ---- tensor_build.cu ----
struct BuildGeom {
    int nx, ny, nz, log2nx, log2ny;
    double dx, dy;
    const double* dz;      // host
    int tile_k;
    long long n_k, n_k_padded;
    int prec;              // hfft_precision
    int num_sms;
    // deduplicated bank: host tables pair -> class [nz*nz], class -> representative pair
    // i*nz+j [n_classes]; pair_class == nullptr: one slot per pair (class = i*nz+j)
    bool mirror = false;   // bank entry p = kx * (ny + 1) + t, t = 0..ny, serves ky = t and ky = 2ny - t; tile_k / 2 per tile
    bool recip = false;    // bank value of the representative pair (p, q), p <= q, is multiplied by dz_p
    bool symv = false;     // recip in the symv layout (symv_layout.h): tile_k / 2 entries per CTA tile of kSymvWarps units
    size_t symv_bank_bytes = 0;
    const int* pair_class = nullptr;
    const int* class_rep = nullptr;
    int n_classes = 0;
};
// tensor classes of the layer pairs: pairs with identical (dz_i, dz_j, zeta_i - zeta_j) share one tensor
void pair_classes(int nz, const double* dz, std::vector<int>& cls, std::vector<int>& rep, bool& toeplitz);
size_t build_scratch_bytes(const BuildGeom& g);
// fills `bank` (plan precision); fp64 tables on device: tw2nx (2nx entries) and the per-thread
// tables of the length-nx and length-2ny row transforms.  changed < 0: every layer pair; else only
// the pairs whose tensor depends on the thickness of layer `changed` (hfft_update_dz)
cudaError_t build_bank(const BuildGeom& g, void* bank, void* scratch, const void* tw2nx_f64, const void* twt_nx_f64,
                       const void* twt_2ny_f64, int changed, cudaStream_t st, std::string& err);

}  // namespace hfft
