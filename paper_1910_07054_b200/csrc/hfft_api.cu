// hfft_api.cu -- the C ABI declared in include/hfft.h: plan object, argument checks, twiddle
// tables, stage orchestration.  No arithmetic of the method lives here except the twiddle table.
#include <math.h>
#include <string.h>

#include <new>

#include "hfft_internal.h"
#include "symv_layout.h"

using namespace hfft;

namespace {
thread_local std::string g_create_error;
constexpr int kMaxProfileCalls = 256;
const char* kPipeBusy =
    ": evaluations of hfft_demag_host_async are outstanding (they use the plan's spectra and bank); call hfft_host_join first";
}  // namespace

struct hfft_plan {
    int nx = 0, ny = 0, nz = 0, batch = 1, log2nx = 0, log2ny = 0;
    hfft_precision prec = HFFT_F32;
    double dx = 0, dy = 0;
    std::vector<double> dz;
    int device = 0, num_sms = 0;
    int tile_k = 0;
    long long n_k = 0, n_k_padded = 0, n_tiles = 0;
    size_t elem = 4;
    size_t bank_bytes = 0, ws_bytes = 0;
    size_t ws_xhat = 0, ws_spec = 0;                 // offsets into the workspace
    // host paths: staging copies of m and h (two slots for the pipelined form), allocated on the first
    // hfft_demag_host / hfft_demag_host_async call -- callers of the device path never pay for them
    void* stage = nullptr;
    size_t stage_bytes = 0;                          // of one buffer; layout m, h, m2, h2
    bool pipe_unjoined = false;                      // hfft_demag_host_async issued since the last hfft_host_join
    // hfft_demag_host_async: copy-in, compute and copy-out streams, per staging slot events
    cudaStream_t s_h2d = nullptr, s_comp = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_user = nullptr, ev_h2d[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr},
                ev_d2h[2] = {nullptr, nullptr};
    unsigned long long pipe_calls = 0;
    void *bank = nullptr, *ws = nullptr;
    bool own_bank = false, own_ws = false, built = false;
    // tw_x: exp(-2 pi i t / 2nx), 2nx entries; twt_x / twt_y: per-thread tables of the length-nx and
    // length-2ny row transforms (fft.cuh).  *64: fp64 copies for the setup (aliases for an fp64 plan).
    void *tw_x = nullptr, *twt_x = nullptr, *twt_y = nullptr;
    void *tw_x64 = nullptr, *twt_x64 = nullptr, *twt_y64 = nullptr;
    double* sums = nullptr;                          // hfft_plan_set_reduction: [B][3][nz][2] on device
    // tensor classes (hfft_plan_set_dedup): pair -> class, class -> representative pair i*nz+j
    int dedup_mode = 1;                              // 0 off, 1 auto, 2 on, 3 z-FFT (Eq.25)
    bool dedup = false, toeplitz = false, class_kernel = false;
    int recip_mode = 2;                              // hfft_plan_set_recip: 0 off, 1 on, 2 automatic
    bool recip = false;                              // bank holds dz_p R_pq for one orientation of every pair (with the mirror storage)
    bool symv = false;                               // ... in the symv layout, read once by coupling_symv_kernel
    std::vector<int> recip_cls, recip_rep;           // pair -> slot of the unordered pair; slot -> p*nz+q (p <= q)
    void* d_invdz = nullptr;                         // 1 / dz_i, plan precision (recip)
    int fuse_mode = 1;                               // hfft_plan_set_fusion: 0 off, 1 automatic (small grids), 2 wherever it fits
    bool fused = false;                              // S2 + S3 + S4 in one kernel (fused_ycy.cu)
    int mirror_mode = 1;                             // hfft_plan_set_mirror: 0 off, 1 automatic
    bool mirror = false;                             // spectrum in the mirror layout, half bank (coupling_kernel MIR)
    long long n_slots = 0;                           // spectrum slots per plane before padding
    bool zfft = false;                               // equal thicknesses: z-convolution by FFT (coupling_zfft.cu)
    int log2lz = 0;
    void* d_twz = nullptr;                           // exp(-2 pi i n / Lz), plan precision
    int n_classes = 0;                               // distinct tensors among the nz^2 pairs
    std::vector<int> pair_class, class_rep;
    unsigned short* d_cls = nullptr;                 // device copy of pair_class (dedup only)
    bool profiling = false;
    int prof_calls = 0;
    std::vector<cudaEvent_t> prof_events;            // (HFFT_NUM_STAGES + 1) per call
    std::string error;
};

// ---- scratch of hfft_update_dz_static (hfft.h) ----
// A fixed array in this translation unit's device image: it exists on every device that loads the image and is never
// freed.  In HOST code the name below is only a handle for the runtime, not a device address -- a kernel handed
// `g_static_scratch` itself would fault (or, where the GPU can reach host memory, quietly work on the wrong bytes).
// The address that kernels can use comes from cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[HFFT_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kMaxCachedDevices = 64;
std::mutex g_static_mu;                                  // held for a whole hfft_update_dz_static call
void* g_static_addr[kMaxCachedDevices] = {};             // device ordinal -> address of g_static_scratch there

// Device address of the scratch array on the CURRENT device `dev`; g_static_mu must be held.
cudaError_t static_scratch_address(int dev, void** out) {
    if (dev >= 0 && dev < kMaxCachedDevices && g_static_addr[dev]) { *out = g_static_addr[dev]; return cudaSuccess; }
    void* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!ptr || ((size_t)ptr & 255)) return cudaErrorInvalidSymbol;
    if (dev >= 0 && dev < kMaxCachedDevices) g_static_addr[dev] = ptr;
    *out = ptr;
    return cudaSuccess;
}
}  // namespace

static hfft_status fail(hfft_plan* p, hfft_status s, const std::string& msg) {
    if (p) p->error = msg; else g_create_error = msg;
    return s;
}
static hfft_status fail_cuda(hfft_plan* p, const char* what, cudaError_t e) {
    return fail(p, HFFT_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
static bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
static int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }

// exp(-2 pi i t / N), t in [0, N): the angle is reduced to the first octant in integers so that
// every entry is the correctly rounded image of an exact rational multiple of pi
static void twiddle_table(int N, std::vector<double>& re, std::vector<double>& im) {
    re.resize(N); im.resize(N);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int t = 0; t < N; ++t) {
        // angle = 2 pi t / N = (pi/4) * (8 t / N); octant o = floor(8t/N), remainder r/N of an octant
        long long num = 8LL * t;
        int o = (int)(num / N);
        long long r = num % N;                     // angle = (o + r/N) * pi/4
        long double c, s;
        // within an octant use the smaller of r/N and 1 - r/N
        bool flip = (o & 1) != 0;
        long double frac = flip ? (long double)(N - r) / N : (long double)r / N;   // in [0, 1]
        long double a = frac * (pi / 4);
        long double ca = cosl(a), sa = sinl(a);
        if (r == 0) { ca = flip ? sqrtl(0.5L) : 1.0L; sa = flip ? sqrtl(0.5L) : 0.0L; }
        // base angle of the octant pair: q = o / 2 quarter turns (+ an eighth handled by flip)
        // angle = q * pi/2 + (flip ? pi/2 - a : a)
        long double cb = flip ? sa : ca, sb = flip ? ca : sa;   // cos/sin of the in-quadrant angle
        switch ((o / 2) & 3) {
            case 0: c = cb; s = sb; break;
            case 1: c = -sb; s = cb; break;
            case 2: c = -cb; s = -sb; break;
            default: c = sb; s = -cb; break;
        }
        re[t] = (double)c;
        im[t] = (double)(-s);
    }
}

// Per-thread twiddle table of the length-2^log2N row transform, in the order the kernels consume it
// (fft.cuh, RowFFT): stages after the first; radix 2^lr, U = R / radix butterflies per thread;
// slot (stage, u, t) holds, for thread j < TPR, exp(-2 pi i t k / (N_s radix)), k = (j + u TPR) mod N_s.
static void thread_twiddle_table(int log2N, std::vector<double>& re, std::vector<double>& im) {
    const int N = 1 << log2N, log2R = log2N < 3 ? log2N : 3, R = 1 << log2R, TPR = N / R;
    std::vector<double> tr, ti;
    twiddle_table(N, tr, ti);
    re.clear(); im.clear();
    for (int lns = log2R; lns < log2N;) {
        const int lr = (log2N - lns >= 3) ? 3 : log2N - lns;
        const int rad = 1 << lr, U = R / rad, NS = 1 << lns;
        for (int u = 0; u < U; ++u)
            for (int t = 1; t < rad; ++t)
                for (int j = 0; j < TPR; ++j) {
                    const long long k = (j + u * TPR) & (NS - 1);
                    const long long idx = (t * k * (N >> (lns + lr))) % N;
                    re.push_back(tr[idx]); im.push_back(ti[idx]);
                }
        lns += lr;
    }
    if (re.empty()) { re.push_back(1.0); im.push_back(0.0); }   // single-stage transforms read nothing
}

static cudaError_t upload_complex(const std::vector<double>& re, const std::vector<double>& im, bool f32, void** out) {
    const size_t n = re.size();
    cudaError_t e;
    if (f32) {
        std::vector<float> h(2 * n);
        for (size_t t = 0; t < n; ++t) { h[2 * t] = (float)re[t]; h[2 * t + 1] = (float)im[t]; }
        if ((e = cudaMalloc(out, h.size() * sizeof(float))) != cudaSuccess) return e;
        return cudaMemcpy(*out, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice);
    }
    std::vector<double> h(2 * n);
    for (size_t t = 0; t < n; ++t) { h[2 * t] = re[t]; h[2 * t + 1] = im[t]; }
    if ((e = cudaMalloc(out, h.size() * sizeof(double))) != cudaSuccess) return e;
    return cudaMemcpy(*out, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice);
}
static cudaError_t upload_twiddles(int N, bool f32, void** out) {
    std::vector<double> re, im;
    twiddle_table(N, re, im);
    return upload_complex(re, im, f32, out);
}
static cudaError_t upload_thread_twiddles(int log2N, bool f32, void** out) {
    std::vector<double> re, im;
    thread_twiddle_table(log2N, re, im);
    return upload_complex(re, im, f32, out);
}

static BuildGeom make_geom(const hfft_plan* p) {
    BuildGeom g{p->nx, p->ny, p->nz, p->log2nx, p->log2ny, p->dx, p->dy, p->dz.data(),
                p->tile_k, p->n_k, p->n_k_padded, p->prec, p->num_sms};
    g.mirror = p->mirror;
    g.symv = p->symv; g.symv_bank_bytes = p->symv ? p->bank_bytes : 0;
    if (p->dedup) { g.pair_class = p->pair_class.data(); g.class_rep = p->class_rep.data(); g.n_classes = p->n_classes; }
    if (p->recip) {
        g.pair_class = p->recip_cls.data(); g.class_rep = p->recip_rep.data(); g.n_classes = (int)p->recip_rep.size();
        g.recip = true;
    }
    return g;
}

// 1 / dz_i in the plan precision (reciprocity storage: H_i = (1 / dz_i) sum_j S_ij M_j)
static cudaError_t upload_inv_dz(hfft_plan* p) {
    cudaError_t e;
    if (!p->d_invdz && (e = cudaMalloc(&p->d_invdz, p->nz * p->elem)) != cudaSuccess) return e;
    std::vector<float> f(p->nz);
    std::vector<double> d(p->nz);
    for (int k = 0; k < p->nz; ++k) { d[k] = 1.0 / p->dz[k]; f[k] = (float)d[k]; }
    return cudaMemcpy(p->d_invdz, p->elem == 4 ? (const void*)f.data() : (const void*)d.data(), p->nz * p->elem,
                      cudaMemcpyHostToDevice);
}

static void plan_sizes(hfft_plan* p) {
    const size_t e = p->elem;
    p->n_k = 2LL * p->ny * (p->nx + 1);
    const int wide = 32 * (int)(16 / e);
    const bool big = p->n_k / wide >= 2LL * (p->num_sms > 0 ? p->num_sms : 148);
    // ky-mirror storage (the spectra are even or odd in ky): where the plain streaming kernel would run
    // with wide tiles (mode 2: on any grid) it reads one bank value per pair (ky, 2ny - ky); the spectrum rows then
    // have 2ny + 2 slots (fft_kernels.cu ypos).  Tiles of 64 slots = 32 bank entries, one per lane, in both
    // precisions: measured faster than 128-slot tiles in fp32 (B200, C4: 1.11 vs 1.28 ms, C3: 0.084 vs 0.098 ms --
    // two or more CTAs with their M^ tiles share an SM).
    const bool mirror_ok = p->mirror_mode >= 1 && (big || p->mirror_mode == 2) && p->ny >= 2 &&
                           !coupling_batched_applies(p->nz, p->batch, e) && coupling_smem_bytes(p->nz, 64, e) <= 200 * 1024;
    // equal thicknesses: the z-convolution by FFT (Eq.25) where it applies, from 16 layers on
    // (below that the explicit Toeplitz sum does less work)
    p->zfft = p->toeplitz && coupling_zfft_applies(p->nz, e, &p->log2lz) &&
              (p->dedup_mode == 3 || (p->dedup_mode == 1 && p->nz >= 16));
    // deduplicated bank (mode 2: always).  Automatic mode: once at most half of the pairs carry a tensor of their own
    // AND the class path is the faster one.  Measured on B200 at 256 x 256 fp32 (profiles/r02_scaling_nz.md): the z-FFT
    // and the Toeplitz window kernel always win; the generic class kernel (bank tile in shared memory, bound by its
    // bandwidth) wins up to 8 layers and loses to the mirror / reciprocity bank from 16 on (nz = 32: 0.35 vs 0.28 ms),
    // the class-indexed streaming fallback (tile too large for shared memory) loses by 1.5-2x (nz = 64: 1.53 vs 0.79 ms)
    // -- so those two are chosen only where the mirror storage does not apply (small grids, nz > 133 in fp32).
    const bool few = 2 * p->n_classes <= p->nz * p->nz;
    const bool fits = coupling_class_smem_bytes(p->nz, p->n_classes, p->toeplitz, e) <= 220 * 1024;
    bool auto_dedup = few;
    if (few && mirror_ok && !p->zfft) {
        if (!fits) auto_dedup = false;                               // streaming fallback
        else if (!p->toeplitz && p->nz > 8) auto_dedup = false;      // generic class kernel
    }
    p->dedup = p->dedup_mode == 2 || (p->dedup_mode == 1 && auto_dedup);
    if (p->zfft) p->dedup = true;
    p->class_kernel = p->dedup && !p->zfft && fits;
    // wide tiles (128-bit bank loads per lane) once there are enough of them to fill the chip twice
    p->tile_k = big ? wide : 32;
    while (p->tile_k > 32 && coupling_smem_bytes(p->nz, p->tile_k, e) > 200 * 1024) p->tile_k /= 2;
    if (p->tile_k != wide) p->tile_k = 32;
    if (!p->dedup && coupling_batched_applies(p->nz, p->batch, e)) p->tile_k = 32;
    if (p->class_kernel || p->zfft) p->tile_k = 32;
    p->mirror = mirror_ok && !p->dedup;
    if (p->mirror) p->tile_k = 64;
    // S2 + S3 + S4 fused (fused_ycy.cu): plain bank in 32-wavevector tiles, the kx column of all planes in one CTA's
    // shared memory.  Automatic on the small grids only (those that do not fill the chip with wide tiles: they are bound
    // by launches, not bytes -- B200, 64 x 64 x 6: 22.8 -> see DESIGN.md 8); mode 2 forces it wherever it fits.
    {
        const size_t fs = fused_ycy_smem_bytes(p->log2ny + 1, p->nz, e);
        p->fused = p->fuse_mode >= 1 && !p->dedup && !p->zfft &&
                   (p->fuse_mode == 2 || !coupling_batched_applies(p->nz, p->batch, e)) && fs > 0 && fs <= 222 * 1024 &&
                   (p->fuse_mode == 2 ? p->mirror_mode != 2 : !p->mirror && !big && fused_ycy_pays(p->log2ny + 1, p->nz, e));
        if (p->fused) { p->mirror = false; p->tile_k = 32; }
    }
    // reciprocity storage on top of the mirror storage.  fp32, nz <= 64: the symv layout, every block read
    // once and used for both of its layer pairs (coupling_symv.cu) -- automatic from 8 layers on where it streams at
    // least 30 % fewer bytes than the mirror bank (the layout pads nz to whole strips of 4, the strips to a power of two);
    // otherwise (mode 1 only) the p <= q storage read through the class table of the streaming kernel.
    p->symv = false;
    if (p->mirror && p->recip_mode >= 1 && coupling_symv_applies(p->nz, e)) {
        const SymvGeom G = symv_geom(p->nz);
        const bool wins = p->nz >= 8 && symv_pairs_per_entry(G) * 10 <= (long long)p->nz * p->nz * 7;
        p->symv = p->recip_mode == 1 || wins;
    }
    p->recip = p->symv || (p->mirror && p->recip_mode == 1 && p->nz >= 2 && p->nz * (p->nz + 1) / 2 <= 65535);
    p->recip_cls.clear(); p->recip_rep.clear();
    if (p->recip) {
        // slot of the unordered pair and its stored orientation (p, q): S_pq = dz_p R_pq; (q, p) is its transpose
        const int nz = p->nz;
        const SymvGeom G = symv_geom(nz);
        p->recip_cls.assign((size_t)nz * nz, 0);
        for (int a = 0; a < nz; ++a)
            for (int b = a; b < nz; ++b) {
                const int slot = (int)p->recip_rep.size();
                const bool swap = p->symv && symv_pos(G, a, b).transposed;
                p->recip_rep.push_back(swap ? b * nz + a : a * nz + b);
                p->recip_cls[(size_t)a * nz + b] = p->recip_cls[(size_t)b * nz + a] = slot;
            }
    }
    if (p->symv) p->tile_k = 2 * coupling_symv_tile_entries(p->nz);
    p->n_slots = p->mirror ? (long long)(p->nx + 1) * (2 * p->ny + 2) : p->n_k;
    p->n_tiles = (p->n_slots + p->tile_k - 1) / p->tile_k;
    p->n_k_padded = p->n_tiles * p->tile_k;
    const size_t slots = p->zfft ? (((size_t)1 << p->log2lz) / 2 + 1)          // S(k, kz), kz = 0 .. Lz / 2 (coupling_zfft.cu)
                         : (p->recip ? (size_t)p->nz * (p->nz + 1) / 2 : (p->dedup ? p->n_classes : p->nz * p->nz));
    p->bank_bytes = (size_t)6 * slots * (size_t)(p->mirror ? p->n_k_padded / 2 : p->n_k_padded) * e;
    if (p->symv) p->bank_bytes = coupling_symv_bank_bytes(p->nz, p->n_tiles);
    const size_t planes = (size_t)3 * p->nz * p->batch;
    auto al = [](size_t v) { return (v + 255) & ~(size_t)255; };
    size_t o = 0;
    p->ws_xhat = o;    o += al(planes * (size_t)p->ny * (p->nx + 1) * 2 * e);
    p->ws_spec = o;    o += al(planes * (size_t)p->n_k_padded * 2 * e);
    p->ws_bytes = o;
    p->stage_bytes = al(planes * (size_t)p->ny * p->nx * e);
}

extern "C" {

const char* hfft_version(void) { return "hfft 0.4 sm_100a"; }

const char* hfft_last_error(const hfft_plan* plan) { return plan ? plan->error.c_str() : g_create_error.c_str(); }

hfft_status hfft_plan_create(hfft_plan** out, int nx, int ny, int nz, double dx, double dy, const double* dz,
                             hfft_precision precision) {
    if (!out) return fail(nullptr, HFFT_EINVAL, "hfft_plan_create: out is NULL");
    *out = nullptr;
    if (!dz) return fail(nullptr, HFFT_EINVAL, "hfft_plan_create: dz is NULL");
    if (nx < 2 || ny < 2 || nz < 1) return fail(nullptr, HFFT_EINVAL, "hfft_plan_create: need nx, ny >= 2 and nz >= 1");
    if (!(dx > 0) || !(dy > 0) || !isfinite(dx) || !isfinite(dy))
        return fail(nullptr, HFFT_EINVAL, "hfft_plan_create: dx, dy must be positive and finite");
    for (int k = 0; k < nz; ++k)
        if (!(dz[k] > 0) || !isfinite(dz[k]))
            return fail(nullptr, HFFT_EINVAL, "hfft_plan_create: every dz[k] must be positive and finite");
    if (precision != HFFT_F32 && precision != HFFT_F64)
        return fail(nullptr, HFFT_EINVAL, "hfft_plan_create: unknown precision");
    if (!is_pow2(nx) || !is_pow2(ny))
        return fail(nullptr, HFFT_EUNSUPPORTED, "hfft_plan_create: nx and ny must be powers of two");
    if (nx > 1024 || ny > 1024) return fail(nullptr, HFFT_EUNSUPPORTED, "hfft_plan_create: nx, ny <= 1024");
    if (nz > HFFT_MAX_NZ) return fail(nullptr, HFFT_EUNSUPPORTED, "hfft_plan_create: nz exceeds HFFT_MAX_NZ");

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(nullptr, "cudaGetDevice (no CUDA device: this library has no CPU path)", e);
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) return fail_cuda(nullptr, "cudaGetDeviceProperties", e);
    if (prop.major != 10)
        return fail(nullptr, HFFT_EUNSUPPORTED, "hfft_plan_create: device is not compute capability 10.x (built for sm_100a)");

    hfft_plan* p = new (std::nothrow) hfft_plan();
    if (!p) return fail(nullptr, HFFT_ENOMEM, "hfft_plan_create: out of host memory");
    p->nx = nx; p->ny = ny; p->nz = nz; p->dx = dx; p->dy = dy; p->prec = precision;
    p->log2nx = ilog2(nx); p->log2ny = ilog2(ny);
    p->dz.assign(dz, dz + nz);
    p->device = dev; p->num_sms = prop.multiProcessorCount;
    p->elem = precision == HFFT_F32 ? 4 : 8;
    pair_classes(nz, p->dz.data(), p->pair_class, p->class_rep, p->toeplitz);
    p->n_classes = (int)p->class_rep.size();
    plan_sizes(p);
    if (coupling_smem_bytes(nz, p->tile_k, p->elem) > 200 * 1024) {
        delete p;
        return fail(nullptr, HFFT_EUNSUPPORTED, "hfft_plan_create: nz too large for the coupling kernel's shared memory");
    }
    *out = p;
    return HFFT_OK;
}

hfft_status hfft_plan_set_batch(hfft_plan* plan, int batch) {
    if (!plan) return HFFT_EINVAL;
    if (batch < 1) return fail(plan, HFFT_EINVAL, "hfft_plan_set_batch: batch < 1");
    if (plan->built || plan->ws) return fail(plan, HFFT_ESTATE, "hfft_plan_set_batch: after build / set_buffers");
    plan->batch = batch;
    plan_sizes(plan);
    return HFFT_OK;
}

hfft_status hfft_plan_set_dedup(hfft_plan* plan, int mode) {
    if (!plan) return HFFT_EINVAL;
    if (mode < 0 || mode > 3) return fail(plan, HFFT_EINVAL, "hfft_plan_set_dedup: mode must be 0, 1, 2 or 3");
    if (plan->built || plan->ws) return fail(plan, HFFT_ESTATE, "hfft_plan_set_dedup: after build / set_buffers");
    if (mode == 3 && !(plan->toeplitz && coupling_zfft_applies(plan->nz, plan->elem, nullptr)))
        return fail(plan, HFFT_EUNSUPPORTED,
                    "hfft_plan_set_dedup: the z-FFT method (mode 3) needs equal layer thicknesses, nz >= 2 and "
                    "nz <= 128 (fp32) / 32 (fp64)");
    plan->dedup_mode = mode;
    plan_sizes(plan);
    return HFFT_OK;
}

hfft_status hfft_plan_set_mirror(hfft_plan* plan, int on) {
    if (!plan) return HFFT_EINVAL;
    if (on < 0 || on > 2) return fail(plan, HFFT_EINVAL, "hfft_plan_set_mirror: 0, 1 or 2");
    if (plan->built || plan->ws) return fail(plan, HFFT_ESTATE, "hfft_plan_set_mirror: after build / set_buffers");
    plan->mirror_mode = on;
    plan_sizes(plan);
    return HFFT_OK;
}

hfft_status hfft_plan_set_fusion(hfft_plan* plan, int mode) {
    if (!plan) return HFFT_EINVAL;
    if (mode < 0 || mode > 2) return fail(plan, HFFT_EINVAL, "hfft_plan_set_fusion: 0, 1 or 2");
    if (plan->built || plan->ws) return fail(plan, HFFT_ESTATE, "hfft_plan_set_fusion: after build / set_buffers");
    plan->fuse_mode = mode;
    plan_sizes(plan);
    return HFFT_OK;
}

hfft_status hfft_plan_set_recip(hfft_plan* plan, int on) {
    if (!plan) return HFFT_EINVAL;
    if (on < 0 || on > 2) return fail(plan, HFFT_EINVAL, "hfft_plan_set_recip: 0, 1 or 2");
    if (plan->built || plan->ws) return fail(plan, HFFT_ESTATE, "hfft_plan_set_recip: after build / set_buffers");
    plan->recip_mode = on;
    plan_sizes(plan);
    return HFFT_OK;
}

hfft_status hfft_tensor_classes(int nz, const double* dz, int* cls_out, int* n_classes, int* toeplitz) {
    if (!dz || !cls_out || !n_classes || !toeplitz || nz < 1 || nz > HFFT_MAX_NZ) return HFFT_EINVAL;
    for (int k = 0; k < nz; ++k)
        if (!(dz[k] > 0) || !isfinite(dz[k])) return HFFT_EINVAL;
    std::vector<int> cls, rep;
    bool toep = false;
    pair_classes(nz, dz, cls, rep, toep);
    for (size_t x = 0; x < cls.size(); ++x) cls_out[x] = cls[x];
    *n_classes = (int)rep.size();
    *toeplitz = toep ? 1 : 0;
    return HFFT_OK;
}

hfft_status hfft_plan_info(const hfft_plan* plan, hfft_info* info) {
    if (!plan || !info) return HFFT_EINVAL;
    info->nx = plan->nx; info->ny = plan->ny; info->nz = plan->nz; info->batch = plan->batch;
    info->precision = plan->prec; info->tile_k = plan->tile_k;
    info->n_k = plan->n_k; info->n_k_padded = plan->n_k_padded;
    info->bank_bytes = plan->bank_bytes; info->workspace_bytes = plan->ws_bytes;
    BuildGeom g = make_geom(plan);
    info->setup_scratch_bytes = build_scratch_bytes(g);
    info->launches_per_demag = plan->fused ? 3 : HFFT_NUM_STAGES;
    info->fused = plan->fused ? 1 : 0;
    info->built = plan->built ? 1 : 0;
    info->n_classes = plan->n_classes;
    info->mirror = plan->mirror ? (plan->symv ? 3 : (plan->recip ? 2 : 1)) : 0;
    info->dedup = plan->zfft ? 4 : (plan->dedup ? (plan->class_kernel ? (plan->toeplitz ? 3 : 2) : 1) : 0);
    return HFFT_OK;
}

size_t hfft_bank_bytes(const hfft_plan* plan) { return plan ? plan->bank_bytes : 0; }

size_t hfft_workspace_bytes(const hfft_plan* plan) { return plan ? plan->ws_bytes : 0; }

hfft_status hfft_plan_set_buffers(hfft_plan* plan, void* bank, void* workspace) {
    if (!plan) return HFFT_EINVAL;
    if (!bank || !workspace) return fail(plan, HFFT_EINVAL, "hfft_plan_set_buffers: NULL buffer");
    if (((size_t)bank & 255) || ((size_t)workspace & 255))
        return fail(plan, HFFT_EINVAL, "hfft_plan_set_buffers: buffers must be 256-byte aligned");
    if (plan->built) return fail(plan, HFFT_ESTATE, "hfft_plan_set_buffers: after hfft_build_tensor");
    plan->bank = bank; plan->ws = workspace; plan->own_bank = plan->own_ws = false;
    return HFFT_OK;
}

hfft_status hfft_build_tensor(hfft_plan* plan, void* stream) {
    if (!plan) return HFFT_EINVAL;
    // a rebuild rewrites the bank (and clears the spectra) on the caller's stream while the pipeline's own compute
    // stream may still be reading them
    if (plan->pipe_unjoined) return fail(plan, HFFT_ESTATE, std::string("hfft_build_tensor") + kPipeBusy);
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if ((e = cudaSetDevice(plan->device)) != cudaSuccess) return fail_cuda(plan, "cudaSetDevice", e);
    if (!plan->bank) {
        if ((e = cudaMalloc(&plan->bank, plan->bank_bytes)) != cudaSuccess)
            return fail(plan, HFFT_ENOMEM, std::string("cudaMalloc(bank): ") + cudaGetErrorString(e));
        plan->own_bank = true;
    }
    if (!plan->ws) {
        if ((e = cudaMalloc(&plan->ws, plan->ws_bytes)) != cudaSuccess)
            return fail(plan, HFFT_ENOMEM, std::string("cudaMalloc(workspace): ") + cudaGetErrorString(e));
        plan->own_ws = true;
    }
    // padded wavevectors of the spectra must hold finite values
    if ((e = cudaMemsetAsync(plan->ws, 0, plan->ws_bytes, st)) != cudaSuccess) return fail_cuda(plan, "cudaMemsetAsync", e);
    // every table is guarded on its own: a build that failed half-way through the uploads is retried cleanly
    if (!plan->tw_x64 && (e = upload_twiddles(2 * plan->nx, false, &plan->tw_x64)) != cudaSuccess) return fail_cuda(plan, "twiddles", e);
    if (!plan->twt_x64 && (e = upload_thread_twiddles(plan->log2nx, false, &plan->twt_x64)) != cudaSuccess) return fail_cuda(plan, "twiddles", e);
    if (!plan->twt_y64 && (e = upload_thread_twiddles(plan->log2ny + 1, false, &plan->twt_y64)) != cudaSuccess) return fail_cuda(plan, "twiddles", e);
    if (plan->prec == HFFT_F32) {
        if (!plan->tw_x && (e = upload_twiddles(2 * plan->nx, true, &plan->tw_x)) != cudaSuccess) return fail_cuda(plan, "twiddles", e);
        if (!plan->twt_x && (e = upload_thread_twiddles(plan->log2nx, true, &plan->twt_x)) != cudaSuccess) return fail_cuda(plan, "twiddles", e);
        if (!plan->twt_y && (e = upload_thread_twiddles(plan->log2ny + 1, true, &plan->twt_y)) != cudaSuccess) return fail_cuda(plan, "twiddles", e);
    } else {
        plan->tw_x = plan->tw_x64; plan->twt_x = plan->twt_x64; plan->twt_y = plan->twt_y64;
    }
    if (plan->recip && (e = upload_inv_dz(plan)) != cudaSuccess) return fail_cuda(plan, "1/dz table", e);
    if ((plan->dedup || plan->recip) && !plan->d_cls) {
        const std::vector<int>& tab = plan->recip ? plan->recip_cls : plan->pair_class;
        std::vector<unsigned short> c16(tab.begin(), tab.end());
        if ((e = cudaMalloc(&plan->d_cls, c16.size() * sizeof(unsigned short))) != cudaSuccess)
            return fail(plan, HFFT_ENOMEM, std::string("cudaMalloc(class table): ") + cudaGetErrorString(e));
        if ((e = cudaMemcpy(plan->d_cls, c16.data(), c16.size() * sizeof(unsigned short), cudaMemcpyHostToDevice)) != cudaSuccess)
            return fail_cuda(plan, "cudaMemcpy(class table)", e);
    }
    BuildGeom g = make_geom(plan);
    void* scratch = nullptr;
    const size_t sb = build_scratch_bytes(g);
    if ((e = cudaMalloc(&scratch, sb)) != cudaSuccess)
        return fail(plan, HFFT_ENOMEM, std::string("cudaMalloc(setup scratch): ") + cudaGetErrorString(e));
    std::string msg;
    if (!plan->zfft) {
        e = build_bank(g, plan->bank, scratch, plan->tw_x64, plan->twt_x64, plan->twt_y64, -1, st, msg);
    } else {
        // Toeplitz classes in fp64, plain layout [d][6][n_k_padded] (one "tile" of n_k_padded wavevectors), then their
        // z-DFT into the bank S(k, kz)
        const int LZ = 1 << plan->log2lz;
        void *cls64 = nullptr, *twz64 = nullptr;
        BuildGeom g2 = g;
        g2.prec = HFFT_F64;
        g2.tile_k = (int)plan->n_k_padded;
        e = cudaMalloc(&cls64, (size_t)plan->nz * 6 * plan->n_k_padded * sizeof(double));
        if (e == cudaSuccess) e = upload_twiddles(LZ, false, &twz64);
        if (e == cudaSuccess && !plan->d_twz) e = upload_twiddles(LZ, plan->prec == HFFT_F32, &plan->d_twz);
        if (e != cudaSuccess) msg = std::string("z-FFT setup buffers: ") + cudaGetErrorString(e);
        if (e == cudaSuccess) e = build_bank(g2, cls64, scratch, plan->tw_x64, plan->twt_x64, plan->twt_y64, -1, st, msg);
        if (e == cudaSuccess) {
            e = launch_zdft_bank(plan->bank, (const double*)cls64, twz64, plan->nz, plan->log2lz, plan->n_k,
                                 plan->n_k_padded, plan->n_k_padded, plan->prec, st);
            if (e != cudaSuccess) msg = std::string("zdft_bank_kernel: ") + cudaGetErrorString(e);
        }
        cudaStreamSynchronize(st);
        if (cls64) cudaFree(cls64);
        if (twz64) cudaFree(twz64);
    }
    cudaError_t e2 = cudaStreamSynchronize(st);
    cudaFree(scratch);
    if (e != cudaSuccess) return fail(plan, HFFT_ECUDA, "hfft_build_tensor: " + msg);
    if (e2 != cudaSuccess) return fail_cuda(plan, "hfft_build_tensor: cudaStreamSynchronize", e2);
    plan->built = true;
    return HFFT_OK;
}

}  // extern "C"

template <typename T>
static hfft_status demag_impl(hfft_plan* p, const void* m, const double* Ms, void* h, cudaStream_t st) {
    unsigned char* ws = static_cast<unsigned char*>(p->ws);
    const int planes = 3 * p->nz * p->batch;
    void* xhat = ws + p->ws_xhat;
    void* spec = ws + p->ws_spec;
    cudaEvent_t* ev = nullptr;
    if (p->profiling) {
        if (p->prof_calls >= kMaxProfileCalls) return fail(p, HFFT_ESTATE, "hfft_demag: profile buffer full; call hfft_profile_read");
        ev = p->prof_events.data() + (size_t)p->prof_calls * (HFFT_NUM_STAGES + 1);
    }
    cudaError_t e;
#define STAGE(idx, call)                                                            \
    if (ev && (e = cudaEventRecord(ev[idx], st)) != cudaSuccess) return fail_cuda(p, "cudaEventRecord", e); \
    if ((e = (call)) != cudaSuccess) return fail_cuda(p, #call, e);
    STAGE(0, (launch_fftx_fwd<T, true>((const T*)m, xhat, p->log2nx, planes, p->ny, p->nz, Ms, p->tw_x, p->twt_x,
                                       p->num_sms, st)))
    // the z components are rotated by i on the k side (real form R6) except in the z-FFT mode
    const int nz_rot = p->zfft ? 0 : p->nz;
    if (p->fused) {
        // S2 + S3 + S4 in one launch; the profile charges it to the coupling stage (the two y stages read 0)
        if (ev && ((e = cudaEventRecord(ev[1], st)) != cudaSuccess || (e = cudaEventRecord(ev[2], st)) != cudaSuccess))
            return fail_cuda(p, "cudaEventRecord", e);
        if ((e = launch_fused_ycy<T>(xhat, p->bank, p->nx, p->log2ny + 1, p->nz, p->batch, p->twt_y, p->num_sms, st)) != cudaSuccess)
            return fail_cuda(p, "launch_fused_ycy", e);
        if (ev && (e = cudaEventRecord(ev[3], st)) != cudaSuccess) return fail_cuda(p, "cudaEventRecord", e);
    } else {
    STAGE(1, (launch_ffty_fwd<T, true>(xhat, spec, p->nx, p->log2ny + 1, planes, nz_rot, p->n_k_padded, p->twt_y,
                                       p->num_sms, st, p->mirror ? 1 : 0)))
    CouplingArgs ca{p->bank, spec, p->nz, p->batch, p->tile_k, p->n_tiles, p->n_k_padded,
                    p->recip ? (int)p->recip_rep.size() : (p->dedup ? p->n_classes : p->nz * p->nz),
                    (p->dedup || p->recip) ? p->d_cls : nullptr, p->class_kernel, p->toeplitz, p->num_sms};
    ca.recip = p->recip; ca.inv_dz = p->d_invdz; ca.symv = p->symv;
    ca.zfft = p->zfft; ca.log2lz = p->log2lz; ca.twz = p->d_twz; ca.mirror = p->mirror;
    STAGE(2, (launch_coupling<T>(ca, st)))
    STAGE(3, (launch_iffty<T>(spec, xhat, p->nx, p->log2ny + 1, planes, nz_rot, p->n_k_padded, p->twt_y, p->num_sms, st,
                              p->mirror ? 1 : 0)))
    }
    if (p->sums && (e = cudaMemsetAsync(p->sums, 0, (size_t)planes * 2 * sizeof(double), st)) != cudaSuccess)
        return fail_cuda(p, "cudaMemsetAsync(sums)", e);
    STAGE(4, (launch_ifftx<T>(xhat, (T*)h, p->log2nx, planes, p->ny, p->tw_x, p->twt_x, p->num_sms, (const T*)m,
                              p->sums, st)))
#undef STAGE
    if (ev) {
        if ((e = cudaEventRecord(ev[HFFT_NUM_STAGES], st)) != cudaSuccess) return fail_cuda(p, "cudaEventRecord", e);
        p->prof_calls++;
    }
    return HFFT_OK;
}

extern "C" {

// argument checks of the device path; shared by hfft_demag and the host paths (which pass their staging buffers)
static hfft_status demag_checked(hfft_plan* plan, const void* m, const double* Ms, void* h, void* stream) {
    if (!m || !h) return fail(plan, HFFT_EINVAL, "hfft_demag: NULL m or h");
    if (((size_t)m & 15) || ((size_t)h & 15)) return fail(plan, HFFT_EINVAL, "hfft_demag: m and h must be 16-byte aligned");
    // S5 reads m (fused reductions) while it writes h: any overlap of the two ranges corrupts, not only m == h
    const size_t bytes = (size_t)3 * plan->nz * plan->batch * plan->ny * plan->nx * plan->elem;
    const size_t ma = (size_t)m, ha = (size_t)h;
    if (ma < ha + bytes && ha < ma + bytes) return fail(plan, HFFT_EINVAL, "hfft_demag: h must not overlap m");
    if (!plan->built) return fail(plan, HFFT_ESTATE, "hfft_demag: call hfft_build_tensor first");
    cudaStream_t st = (cudaStream_t)stream;
    return plan->prec == HFFT_F32 ? demag_impl<float>(plan, m, Ms, h, st) : demag_impl<double>(plan, m, Ms, h, st);
}

hfft_status hfft_demag(hfft_plan* plan, const void* m, const double* Ms, void* h, void* stream) {
    if (!plan) return HFFT_EINVAL;
    if (plan->pipe_unjoined) return fail(plan, HFFT_ESTATE, std::string("hfft_demag") + kPipeBusy);
    return demag_checked(plan, m, Ms, h, stream);
}

hfft_status hfft_plan_set_reduction(hfft_plan* plan, double* sums_device) {
    if (!plan) return HFFT_EINVAL;
    if (((size_t)sums_device & 7)) return fail(plan, HFFT_EINVAL, "hfft_plan_set_reduction: sums must be 8-byte aligned");
    plan->sums = sums_device;
    return HFFT_OK;
}

hfft_status hfft_update_dz(hfft_plan* plan, int k, double dz_new, void* stream) {
    if (!plan) return HFFT_EINVAL;
    if (k < 0 || k >= plan->nz) return fail(plan, HFFT_EINVAL, "hfft_update_dz: layer index out of range");
    if (!(dz_new > 0) || !isfinite(dz_new)) return fail(plan, HFFT_EINVAL, "hfft_update_dz: dz must be positive and finite");
    if (!plan->built) return fail(plan, HFFT_ESTATE, "hfft_update_dz: call hfft_build_tensor first");
    if (plan->pipe_unjoined) return fail(plan, HFFT_ESTATE, std::string("hfft_update_dz") + kPipeBusy);
    if (plan->dedup)
        return fail(plan, HFFT_EUNSUPPORTED, "hfft_update_dz: the bank is deduplicated; create the plan with hfft_plan_set_dedup(plan, 0)");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if ((e = cudaSetDevice(plan->device)) != cudaSuccess) return fail_cuda(plan, "cudaSetDevice", e);
    // the new thickness is committed only once the rebuild has gone through: a failure leaves dz as it was and the
    // plan unbuilt (the bank may be half rewritten), never a bank that disagrees with dz
    const double dz_old = plan->dz[k];
    plan->dz[k] = dz_new;
    BuildGeom g = make_geom(plan);
    void* scratch = nullptr;
    if ((e = cudaMalloc(&scratch, build_scratch_bytes(g))) != cudaSuccess) {
        plan->dz[k] = dz_old;                                // nothing was touched: the plan stays built
        return fail(plan, HFFT_ENOMEM, std::string("cudaMalloc(setup scratch): ") + cudaGetErrorString(e));
    }
    std::string msg;
    // reciprocity storage: the stored orientation S_pq = dz_p R_pq of every changed pair is rebuilt (row_runs picks
    // them out of the pair table; the untouched blocks of the symv layout keep their values, no memset); and the
    // 1 / dz table changes
    e = build_bank(g, plan->bank, scratch, plan->tw_x64, plan->twt_x64, plan->twt_y64, k, st, msg);
    if (e == cudaSuccess && plan->recip && (e = upload_inv_dz(plan)) != cudaSuccess) msg = "1/dz table";
    cudaError_t e2 = cudaStreamSynchronize(st);
    cudaFree(scratch);
    if (e != cudaSuccess || e2 != cudaSuccess) {
        plan->dz[k] = dz_old;
        plan->built = false;
        if (e != cudaSuccess) return fail(plan, HFFT_ECUDA, "hfft_update_dz: " + msg);
        return fail_cuda(plan, "hfft_update_dz: cudaStreamSynchronize", e2);
    }
    // the tensor classes of the new stack (hfft_plan_info.n_classes; the bank itself is not deduplicated here)
    pair_classes(plan->nz, plan->dz.data(), plan->pair_class, plan->class_rep, plan->toeplitz);
    plan->n_classes = (int)plan->class_rep.size();
    return HFFT_OK;
}

// hfft_update_dz without device allocation (hfft.h): the rebuild of hfft_update_dz with its scratch in g_static_scratch.
// The existing function is left as it is; this one repeats its few lines of orchestration.
hfft_status hfft_update_dz_static(hfft_plan* plan, int k, double dz_new, void* stream) {
    if (!plan) return HFFT_EINVAL;
    if (k < 0 || k >= plan->nz) return fail(plan, HFFT_EINVAL, "hfft_update_dz_static: layer index out of range");
    if (!(dz_new > 0) || !isfinite(dz_new)) return fail(plan, HFFT_EINVAL, "hfft_update_dz_static: dz must be positive and finite");
    if (!plan->built) return fail(plan, HFFT_ESTATE, "hfft_update_dz_static: call hfft_build_tensor first");
    if (plan->pipe_unjoined) return fail(plan, HFFT_ESTATE, std::string("hfft_update_dz_static") + kPipeBusy);
    if (plan->dedup)
        return fail(plan, HFFT_EUNSUPPORTED, "hfft_update_dz_static: the bank is deduplicated; create the plan with hfft_plan_set_dedup(plan, 0)");
    if (plan->recip && !plan->d_invdz) return fail(plan, HFFT_ESTATE, "hfft_update_dz_static: 1/dz table missing; rebuild the plan");
    // the size depends on the grid and the layer count only, not on the thicknesses: check it before anything changes
    {
        const size_t need = build_scratch_bytes(make_geom(plan));
        if (need > (size_t)HFFT_STATIC_SCRATCH_BYTES)
            return fail(plan, HFFT_EUNSUPPORTED,
                        "hfft_update_dz_static: this plan needs " + std::to_string(need) + " bytes of setup scratch, the fixed array holds " +
                            std::to_string((size_t)HFFT_STATIC_SCRATCH_BYTES) + " (HFFT_STATIC_SCRATCH_BYTES); use hfft_update_dz");
    }
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if ((e = cudaSetDevice(plan->device)) != cudaSuccess) return fail_cuda(plan, "cudaSetDevice", e);
    // one rebuild at a time per process: the array is shared by every plan and thread, and the call below ends with
    // a synchronisation of `st`, so nothing of this call is still running when the lock is released
    std::lock_guard<std::mutex> lock(g_static_mu);
    void* scratch = nullptr;
    if ((e = static_scratch_address(plan->device, &scratch)) != cudaSuccess)
        return fail_cuda(plan, "hfft_update_dz_static: cudaGetSymbolAddress(static scratch)", e);
    const double dz_old = plan->dz[k];
    plan->dz[k] = dz_new;
    BuildGeom g = make_geom(plan);
    std::string msg;
    // The array still holds the previous call's intermediates.  build_bank writes every table it reads (interface
    // coordinates, class table, lattice and stencil values, transforms) and clears, on `st`, the real-space planes
    // whose padding must be zero -- the same as with the uninitialised memory cudaMalloc hands out.
    e = build_bank(g, plan->bank, scratch, plan->tw_x64, plan->twt_x64, plan->twt_y64, k, st, msg);
    if (e == cudaSuccess && plan->recip && (e = upload_inv_dz(plan)) != cudaSuccess) msg = "1/dz table";   // d_invdz exists: a copy only
    cudaError_t e2 = cudaStreamSynchronize(st);
    if (e != cudaSuccess || e2 != cudaSuccess) {
        plan->dz[k] = dz_old;
        plan->built = false;
        if (e != cudaSuccess) return fail(plan, HFFT_ECUDA, "hfft_update_dz_static: " + msg);
        return fail_cuda(plan, "hfft_update_dz_static: cudaStreamSynchronize", e2);
    }
    pair_classes(plan->nz, plan->dz.data(), plan->pair_class, plan->class_rep, plan->toeplitz);
    plan->n_classes = (int)plan->class_rep.size();
    return HFFT_OK;
}

// staging buffers of the host paths: m, h, and a second pair for the pipelined form
static hfft_status stage_init(hfft_plan* p) {
    if (p->stage) return HFFT_OK;
    cudaError_t e = cudaMalloc(&p->stage, 4 * p->stage_bytes);
    if (e != cudaSuccess) return fail(p, HFFT_ENOMEM, std::string("cudaMalloc(host-path staging): ") + cudaGetErrorString(e));
    return HFFT_OK;
}

hfft_status hfft_demag_host(hfft_plan* plan, const void* m_host, const double* Ms, void* h_host, void* stream) {
    if (!plan) return HFFT_EINVAL;
    if (!m_host || !h_host) return fail(plan, HFFT_EINVAL, "hfft_demag_host: NULL m or h");
    if (!plan->built) return fail(plan, HFFT_ESTATE, "hfft_demag_host: call hfft_build_tensor first");
    if (plan->pipe_unjoined) return fail(plan, HFFT_ESTATE, std::string("hfft_demag_host") + kPipeBusy);
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if ((e = cudaSetDevice(plan->device)) != cudaSuccess) return fail_cuda(plan, "cudaSetDevice", e);
    hfft_status s = stage_init(plan);
    if (s != HFFT_OK) return s;
    unsigned char* sg = static_cast<unsigned char*>(plan->stage);
    const size_t bytes = (size_t)3 * plan->nz * plan->batch * plan->ny * plan->nx * plan->elem;
    if ((e = cudaMemcpyAsync(sg, m_host, bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess)
        return fail_cuda(plan, "cudaMemcpyAsync(H2D)", e);
    s = demag_checked(plan, sg, Ms, sg + plan->stage_bytes, stream);
    if (s != HFFT_OK) return s;
    if ((e = cudaMemcpyAsync(h_host, sg + plan->stage_bytes, bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return fail_cuda(plan, "cudaMemcpyAsync(D2H)", e);
    return HFFT_OK;
}

static cudaError_t pipe_init(hfft_plan* p) {
    if (p->s_h2d) return cudaSuccess;
    cudaError_t e;
    if ((e = cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking)) != cudaSuccess) return e;
    if ((e = cudaStreamCreateWithFlags(&p->s_comp, cudaStreamNonBlocking)) != cudaSuccess) return e;
    if ((e = cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking)) != cudaSuccess) return e;
    cudaEvent_t* evs[] = {&p->ev_user, &p->ev_h2d[0], &p->ev_h2d[1], &p->ev_comp[0], &p->ev_comp[1], &p->ev_d2h[0],
                          &p->ev_d2h[1]};
    for (cudaEvent_t* ev : evs)
        if ((e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming)) != cudaSuccess) return e;
    return cudaSuccess;
}

hfft_status hfft_demag_host_async(hfft_plan* plan, const void* m_host, const double* Ms, void* h_host, void* stream) {
    if (!plan) return HFFT_EINVAL;
    if (!m_host || !h_host) return fail(plan, HFFT_EINVAL, "hfft_demag_host_async: NULL m or h");
    if (!plan->built) return fail(plan, HFFT_ESTATE, "hfft_demag_host_async: call hfft_build_tensor first");
    cudaError_t e;
    if ((e = cudaSetDevice(plan->device)) != cudaSuccess) return fail_cuda(plan, "cudaSetDevice", e);
    if ((e = pipe_init(plan)) != cudaSuccess) return fail_cuda(plan, "hfft_demag_host_async: streams / events", e);
    hfft_status s0 = stage_init(plan);
    if (s0 != HFFT_OK) return s0;
    unsigned char* sg = static_cast<unsigned char*>(plan->stage);
    const size_t bytes = (size_t)3 * plan->nz * plan->batch * plan->ny * plan->nx * plan->elem;
    const int slot = (int)(plan->pipe_calls & 1);
    void* dm = sg + (size_t)(2 * slot) * plan->stage_bytes;
    void* dh = sg + (size_t)(2 * slot + 1) * plan->stage_bytes;
    const bool reuse = plan->pipe_calls >= 2;        // the slot was used two calls ago
#define HFFT_PIPE(call) if ((e = (call)) != cudaSuccess) return fail_cuda(plan, "hfft_demag_host_async: " #call, e)
    // copy-in: after everything the caller enqueued on `stream` so far, and after the evaluation that last read the slot
    HFFT_PIPE(cudaEventRecord(plan->ev_user, (cudaStream_t)stream));
    HFFT_PIPE(cudaStreamWaitEvent(plan->s_h2d, plan->ev_user, 0));
    if (reuse) HFFT_PIPE(cudaStreamWaitEvent(plan->s_h2d, plan->ev_comp[slot], 0));
    HFFT_PIPE(cudaMemcpyAsync(dm, m_host, bytes, cudaMemcpyHostToDevice, plan->s_h2d));
    HFFT_PIPE(cudaEventRecord(plan->ev_h2d[slot], plan->s_h2d));
    // evaluation: after its copy-in, and after the copy-out that last read the slot's h
    HFFT_PIPE(cudaStreamWaitEvent(plan->s_comp, plan->ev_h2d[slot], 0));
    if (reuse) HFFT_PIPE(cudaStreamWaitEvent(plan->s_comp, plan->ev_d2h[slot], 0));
    hfft_status s = demag_checked(plan, dm, Ms, dh, plan->s_comp);
    if (s != HFFT_OK) return s;
    plan->pipe_unjoined = true;
    HFFT_PIPE(cudaEventRecord(plan->ev_comp[slot], plan->s_comp));
    // copy-out
    HFFT_PIPE(cudaStreamWaitEvent(plan->s_d2h, plan->ev_comp[slot], 0));
    HFFT_PIPE(cudaMemcpyAsync(h_host, dh, bytes, cudaMemcpyDeviceToHost, plan->s_d2h));
    HFFT_PIPE(cudaEventRecord(plan->ev_d2h[slot], plan->s_d2h));
    ++plan->pipe_calls;
    return HFFT_OK;
}

hfft_status hfft_host_join(hfft_plan* plan, void* stream) {
    if (!plan) return HFFT_EINVAL;
    if (plan->pipe_calls == 0) return HFFT_OK;
    cudaError_t e;
    // copy-outs are serialised on one stream: the last one implies all the earlier ones
    HFFT_PIPE(cudaStreamWaitEvent((cudaStream_t)stream, plan->ev_d2h[(plan->pipe_calls - 1) & 1], 0));
#undef HFFT_PIPE
    plan->pipe_unjoined = false;
    return HFFT_OK;
}

hfft_status hfft_profile_enable(hfft_plan* plan, int on) {
    if (!plan) return HFFT_EINVAL;
    if (on && plan->prof_events.empty()) {
        plan->prof_events.resize((size_t)kMaxProfileCalls * (HFFT_NUM_STAGES + 1));
        for (auto& ev : plan->prof_events) {
            cudaError_t e = cudaEventCreate(&ev);
            if (e != cudaSuccess) return fail_cuda(plan, "cudaEventCreate", e);
        }
    }
    plan->profiling = on != 0;
    plan->prof_calls = 0;
    return HFFT_OK;
}

hfft_status hfft_profile_read(hfft_plan* plan, double stage_ms[HFFT_NUM_STAGES], int* calls) {
    if (!plan || !stage_ms || !calls) return HFFT_EINVAL;
    for (int s = 0; s < HFFT_NUM_STAGES; ++s) stage_ms[s] = 0.0;
    *calls = plan->prof_calls;
    if (plan->prof_calls == 0) return HFFT_OK;
    cudaError_t e = cudaEventSynchronize(plan->prof_events[(size_t)plan->prof_calls * (HFFT_NUM_STAGES + 1) - 1]);
    if (e != cudaSuccess) return fail_cuda(plan, "cudaEventSynchronize", e);
    for (int c = 0; c < plan->prof_calls; ++c) {
        cudaEvent_t* ev = plan->prof_events.data() + (size_t)c * (HFFT_NUM_STAGES + 1);
        for (int s = 0; s < HFFT_NUM_STAGES; ++s) {
            float ms = 0.f;
            if ((e = cudaEventElapsedTime(&ms, ev[s], ev[s + 1])) != cudaSuccess) return fail_cuda(plan, "cudaEventElapsedTime", e);
            stage_ms[s] += ms;
        }
    }
    plan->prof_calls = 0;
    return HFFT_OK;
}

hfft_status hfft_read_bank(const hfft_plan* plan, int i, int j, int c, double* out_host) {
    if (!plan || !out_host) return HFFT_EINVAL;
    hfft_plan* p = const_cast<hfft_plan*>(plan);
    if (i < 0 || i >= p->nz || j < 0 || j >= p->nz || c < 0 || c > 5) return fail(p, HFFT_EINVAL, "hfft_read_bank: index out of range");
    if (!p->built) return fail(p, HFFT_ESTATE, "hfft_read_bank: tensor not built");
    if (p->zfft) return fail(p, HFFT_EUNSUPPORTED, "hfft_read_bank: the bank of the z-FFT mode holds S(k, kz), not N_ij(k)");
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return fail_cuda(p, "cudaDeviceSynchronize", e);
    // bank entries per tile; mirror storage: entry kx * (ny + 1) + t serves ky = t and ky = 2ny - t (xy, yz negated)
    const int tk = p->mirror ? p->tile_k / 2 : p->tile_k;
    const long long n_e = p->mirror ? (long long)(p->nx + 1) * (p->ny + 1) : p->n_k;
    // folded Toeplitz classes: the slot holds N_{|i-j|}; xz, yz change sign for i < j
    // reciprocity storage: the slot of the unordered pair holds dz_p R_pq (p <= q); (q, p) is its transpose
    const double unscale = -4.0 * p->nx * p->ny * ((p->dedup && p->toeplitz && i < j && c >= 4) ? -1.0 : 1.0) *
                           (p->recip ? ((i > j && c >= 4) ? -1.0 : 1.0) / p->dz[i] : 1.0);
    if (p->symv) {
        // symv layout: one float per bank entry, strided by the unit's stream (symv_layout.h); the stored orientation
        // holds dz_p R_pq, the other one is its transpose (xz, yz negated)
        const SymvGeom G = symv_geom(p->nz);
        const SymvPos pos = symv_pos(G, i, j);
        const double us = -4.0 * p->nx * p->ny * ((pos.transposed && c >= 4) ? -1.0 : 1.0) / p->dz[i];
        const long long n_units = (n_e + G.EPW - 1) / G.EPW;
        const size_t unit_bytes = (size_t)G.NC * kSymvCoupleBytes;
        std::vector<float> col((size_t)n_units);
        for (int ent = 0; ent < G.EPW; ++ent) {
            const size_t off = (size_t)symv_float_offset(G, pos, ent, c) * sizeof(float);
            e = cudaMemcpy2D(col.data(), sizeof(float), static_cast<unsigned char*>(p->bank) + off, unit_bytes, sizeof(float),
                             (size_t)n_units, cudaMemcpyDeviceToHost);
            if (e != cudaSuccess) return fail_cuda(p, "cudaMemcpy2D(bank)", e);
            for (long long u = 0; u < n_units; ++u) {
                const long long en = u * G.EPW + ent;
                if (en >= n_e) break;
                const double v = (double)col[(size_t)u] * us;
                const long long kx = en / (p->ny + 1);
                const int ty = (int)(en - kx * (p->ny + 1));
                out_host[kx * 2 * p->ny + ty] = v;
                if (ty > 0 && ty < p->ny) out_host[kx * 2 * p->ny + (2 * p->ny - ty)] = (c == 3 || c == 5) ? -v : v;
            }
        }
        return HFFT_OK;
    }
    std::vector<unsigned char> buf((size_t)tk * p->elem);
    for (long long t = 0; t < p->n_tiles; ++t) {
        const size_t ncls = p->recip ? p->recip_rep.size() : (p->dedup ? p->n_classes : (size_t)p->nz * p->nz);
        const size_t slot = p->recip ? p->recip_cls[(size_t)i * p->nz + j]
                                     : (p->dedup ? p->pair_class[(size_t)i * p->nz + j] : (size_t)i * p->nz + j);
        // plain: [c][tk]; mirror: [component pair][lane][2][KB] (tensor_build.cu pack_kernel) -- read the pair's block
        const size_t blk = ((size_t)t * ncls + slot) * 6 * tk;
        const size_t off = (blk + (p->mirror ? (size_t)(c >> 1) * 2 * tk : (size_t)c * tk)) * p->elem;
        const size_t cnt = p->mirror ? 2 * (size_t)tk : (size_t)tk;
        if (buf.size() < cnt * p->elem) buf.resize(cnt * p->elem);
        e = cudaMemcpy(buf.data(), static_cast<unsigned char*>(p->bank) + off, cnt * p->elem, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail_cuda(p, "cudaMemcpy(bank)", e);
        const int KB = tk / 32;
        for (int kk = 0; kk < tk; ++kk) {
            const long long en = t * tk + kk;
            if (en >= n_e) break;
            const int idx = p->mirror ? ((kk / KB) * 2 + (c & 1)) * KB + kk % KB : kk;
            double v = p->elem == 4 ? (double)reinterpret_cast<float*>(buf.data())[idx] : reinterpret_cast<double*>(buf.data())[idx];
            v *= unscale;
            if (!p->mirror) { out_host[en] = v; continue; }
            const long long kx = en / (p->ny + 1);
            const int ty = (int)(en - kx * (p->ny + 1));
            out_host[kx * 2 * p->ny + ty] = v;
            if (ty > 0 && ty < p->ny) out_host[kx * 2 * p->ny + (2 * p->ny - ty)] = (c == 3 || c == 5) ? -v : v;
        }
    }
    return HFFT_OK;
}

hfft_status hfft_destroy(hfft_plan* plan) {
    if (!plan) return HFFT_OK;
    if (plan->own_bank && plan->bank) cudaFree(plan->bank);
    if (plan->own_ws && plan->ws) cudaFree(plan->ws);
    if (plan->prec == HFFT_F32) { cudaFree(plan->tw_x); cudaFree(plan->twt_x); cudaFree(plan->twt_y); }
    cudaFree(plan->tw_x64); cudaFree(plan->twt_x64); cudaFree(plan->twt_y64);
    if (plan->stage) cudaFree(plan->stage);
    if (plan->s_h2d) {
        cudaStreamSynchronize(plan->s_h2d); cudaStreamSynchronize(plan->s_comp); cudaStreamSynchronize(plan->s_d2h);
        cudaStreamDestroy(plan->s_h2d); cudaStreamDestroy(plan->s_comp); cudaStreamDestroy(plan->s_d2h);
        cudaEvent_t evs[] = {plan->ev_user, plan->ev_h2d[0], plan->ev_h2d[1], plan->ev_comp[0], plan->ev_comp[1],
                             plan->ev_d2h[0], plan->ev_d2h[1]};
        for (cudaEvent_t ev : evs) if (ev) cudaEventDestroy(ev);
    }
    if (plan->d_cls) cudaFree(plan->d_cls);
    if (plan->d_twz) cudaFree(plan->d_twz);
    if (plan->d_invdz) cudaFree(plan->d_invdz);
    for (auto& ev : plan->prof_events) cudaEventDestroy(ev);
    delete plan;
    return HFFT_OK;
}

}  // extern "C"
