/*
 * hfft.h -- C ABI of the B200-native hybrid-FFT demagnetization field library.
 *
 * Method: Heistracher et al., "Hybrid FFT algorithm for fast demagnetization
 * field calculations on non-equidistant magnetic layers", arXiv 1910.07054.
 * Citations are PAPER.md:<line> (+ equation); readings A1..A16 are listed in
 * DESIGN.md.
 *
 * What the library computes (Eq.18 with PAPER.md:150 Eq.19):
 *
 *   H_a(a1,a2,i) = - sum_j Ms_j sum_{b1,b2} sum_b N^{ab}_{ij}((a1-b1)dx,(a2-b2)dy) m_b(b1,b2,j)
 *
 * for nz layers of nx x ny cells with common in-plane cell size dx x dy and a
 * per-layer thickness dz[j], N_ij the generalized Newell
 * tensor of two cuboids of unequal thickness (PAPER.md:52 Eq.5, :99 Eq.11,
 * :249-291 Eq.27-31).  It is evaluated with the paper's hybrid scheme
 * (Eq.24): 2-D FFT in the plane (zero-padded to 2nx x 2ny),
 * explicit layer-to-layer convolution along z at every in-plane wavevector,
 * inverse 2-D FFT, crop.
 *
 * Everything runs on ONE CUDA device (sm_100a), in hand-written kernels; there
 * is no cuFFT, no CPU fallback and no collective.  Every call returns a status;
 * nothing throws across this boundary.  A plan is not thread-safe (one host thread
 * at a time per plan); different plans may be used from different host threads and
 * on different devices of one process (the per-kernel launch attributes the library
 * caches are keyed by device and guarded by a mutex).
 *
 * Storage of the spectral tensor bank -- all give the same field, chosen automatically
 * from the geometry, each switchable before hfft_build_tensor:
 *   plain        one entry per (layer pair, wavevector)
 *   ky mirror    hfft_plan_set_mirror: ky and 2ny-ky share an entry (default on large grids)
 *   reciprocity  hfft_plan_set_recip: unordered layer pairs only, every 3 x 3 block read once and
 *                used for both of its pairs (default from 8 layers on where the mirror storage is, fp32)
 *   classes      hfft_plan_set_dedup: one entry per distinct (dz_i, dz_j, Z_ij); for equal
 *                thicknesses the Toeplitz form or the z-convolution by FFT (Eq.25)
 *
 * Array layout (all calls): [B][3][nz][ny][nx], x fastest, component order
 * (x,y,z), element type float (HFFT_F32) or double (HFFT_F64), 16-byte aligned.
 *
 * Environment variables read by the library (A/B measurements only; none is needed for normal use, each is read
 * once per process): HFFT_NO_PDL=1 launches the kernels of an evaluation in plain stream order instead of with
 * programmatic dependent launch; HFFT_ZFFT_FORM=reg|smem forces the register or the shared-memory form of the
 * z-FFT coupling kernel (hfft_plan_set_dedup mode 3) instead of the choice by layer count.  Results do not change.
 */
#ifndef HFFT_H
#define HFFT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hfft_plan hfft_plan; /* opaque */

typedef enum { HFFT_F32 = 0, HFFT_F64 = 1 } hfft_precision;

typedef enum {
    HFFT_OK = 0,
    HFFT_EINVAL = 1,       /* bad argument (null, non-positive or non-finite size, misaligned pointer) */
    HFFT_ENOMEM = 2,       /* device or host allocation failed */
    HFFT_ECUDA = 3,        /* a CUDA runtime call or kernel launch failed; see hfft_last_error */
    HFFT_ESTATE = 4,       /* call out of order (e.g. hfft_demag before hfft_build_tensor) */
    HFFT_EUNSUPPORTED = 5  /* nx or ny not a power of two or above 1024, nz above HFFT_MAX_NZ or too large for the
                              coupling kernel's shared memory, no sm_100 device */
} hfft_status;

#define HFFT_MAX_NZ 256

/* Stage indices of the hot path. */
enum { HFFT_STAGE_FFTX = 0, HFFT_STAGE_FFTY = 1, HFFT_STAGE_COUPLING = 2,
       HFFT_STAGE_IFFTY = 3, HFFT_STAGE_IFFTX = 4, HFFT_NUM_STAGES = 5 };

/* Geometry and derived sizes of a plan (filled by hfft_plan_info). */
typedef struct {
    int nx, ny, nz, batch;
    int precision;            /* hfft_precision */
    int tile_k;               /* wavevectors per bank tile */
    long long n_k;            /* wavevectors in the Hermitian half spectrum: (nx+1) * 2ny */
    long long n_k_padded;     /* spectrum slots per plane: n_k (mirror storage: (nx+1) * (2ny+2)) rounded up to a
                                 multiple of tile_k */
    size_t bank_bytes;        /* spectral tensor bank: 6 * (nz^2 or n_classes) * n_k_padded * sizeof(element);
                                 half of that with mirror storage */
    size_t workspace_bytes;   /* spectra X^, M^ (H^ overwrites M^).  The host paths allocate their staging copies of
                                 m and h themselves, on first use */
    size_t setup_scratch_bytes; /* allocated inside hfft_build_tensor and freed before it returns */
    int launches_per_demag;   /* kernels hfft_demag enqueues per call: 5, or 3 with the fused S2+S3+S4 kernel */
    int built;                /* 1 once hfft_build_tensor has completed */
    int n_classes;            /* bank slots a deduplicated bank needs: distinct tensors among the nz^2 layer pairs;
                                 nz for equal thicknesses (N_ij and N_ji then differ by the sign of xz, yz only) */
    int mirror;               /* 1: ky-mirror storage (hfft_plan_set_mirror): half the bank, spectrum rows of 2ny+2 slots;
                                 2: with reciprocity storage on top (hfft_plan_set_recip): a quarter of the bank, read
                                    through a pair table; 3: reciprocity storage in the block layout of the
                                    symmetric-matvec kernel (every block read once) */
    int dedup;                /* 0: one bank slot per pair; 1: per class, streamed; 2: per class, bank tile in
                                 shared memory; 3: as 2 with Toeplitz classes (equal thicknesses); 4: equal
                                 thicknesses, z-convolution by FFT (Eq.25) */
    int fused;                /* 1: S2 + S3 + S4 run as one kernel (hfft_plan_set_fusion) */
} hfft_info;

/*
 * Create a plan for nz layers of nx x ny cells (common dx, dy;
 * layer k has thickness dz[k]; layers are stacked contiguously in array order,
 * reading A9).  dz is a HOST array of nz doubles and is copied.  Lengths are in
 * any one unit (the tensor depends on ratios only).  Selects device = the
 * current CUDA device.  No device memory is allocated here.
 * Errors: EINVAL (null out/dz, nx,ny < 2, nz < 1, non-positive or non-finite
 * dx, dy, dz[k]); EUNSUPPORTED (nx or ny not a power of two; nx or ny > 1024, the
 * longest row transform the FFT kernels hold in registers and shared memory;
 * nz > HFFT_MAX_NZ; nz so large that the M^ tile of the coupling kernel (3 nz x 32
 * wavevectors) exceeds 200 KB of shared memory, i.e. nz > 256 in fp32 and nz > 133
 * in fp64; device is not compute capability 10.x); ECUDA (no CUDA device); ENOMEM.
 */
hfft_status hfft_plan_create(hfft_plan **out, int nx, int ny, int nz,
                             double dx, double dy, const double *dz, hfft_precision precision);

/* Number of independent magnetisation states per hfft_demag call (default 1;
 * BASELINE config 5 uses 32).  Must be called before hfft_build_tensor /
 * hfft_plan_set_buffers.  Errors: EINVAL (B < 1), ESTATE. */
hfft_status hfft_plan_set_batch(hfft_plan *plan, int batch);

/*
 * Bank deduplication.  N_ij depends on (dz_i, dz_j, zeta_i - zeta_j)
 * alone (Eq.19 with Eq.5/11), so layer pairs that agree in the three
 * share one tensor ("class"): equal thicknesses -- the equidistant case the paper
 * compares against, PAPER.md:182-189 -- give nz classes instead of nz^2 (2nz-1 values
 * of i-j, folded by reciprocity to |i-j|), periodic
 * multilayers a few per period.  The bank then holds one slot per class
 * (info.bank_bytes shrinks by nz^2 / n_classes) and, where a k-tile of it fits in
 * shared memory, the coupling stage stops being HBM-bound (coupling.cu).
 *   mode 0: off (one slot per pair; required for hfft_update_dz)
 *   mode 1: automatic (default): a class path is taken where n_classes <= nz^2 / 2 AND it was measured faster
 *           than the hybrid with its mirror / reciprocity bank: equal thicknesses always (Toeplitz form below 16
 *           layers, mode 3 from 16 on); other repeating stacks up to 8 layers, and beyond that only where the
 *           mirror storage does not apply (small grids; nz > 133 in fp32)
 *   mode 2: on (class kernel; Toeplitz form for equal thicknesses)
 *   mode 3: equal thicknesses only: the z-convolution by FFT of PAPER.md:182 Eq.25 as stage S3
 *           (zero-padded transforms of length 2^ceil(log2 2nz) along z at every in-plane
 *           wavevector); needs 2 <= nz <= 128 (fp32) / 32 (fp64)
 * info.dedup reports the kernel chosen.  Results are those of the plain bank up to summation
 * order.  Must be called before hfft_build_tensor / hfft_plan_set_buffers.
 * Errors: EINVAL (mode outside 0..3), ESTATE, EUNSUPPORTED (mode 3 on unequal thicknesses or
 * outside its nz range).
 */
hfft_status hfft_plan_set_dedup(hfft_plan *plan, int mode);

/*
 * ky-mirror storage of the bank.  The in-plane parities of the tensor
 * components (xx, yy, zz, xz even in Y; xy, yz odd) make their spectra even / odd in
 * ky, so the wavevectors ky and 2ny - ky share one bank entry (xy, yz with opposite
 * sign).  The bank then holds ny + 1 entries per kx instead of 2ny -- half the bytes
 * the HBM-bound coupling stage streams -- and S2 / S4 keep every pair in adjacent
 * spectrum slots.  on = 1 (default): used wherever the plain streaming coupling kernel
 * runs with wide tiles (large grids, no deduplication, not the batched register
 * kernel); on = 0: never; on = 2: also on small grids (wide tiles forced; tests).
 * info.mirror tells which.  Results are those of the plain
 * storage (the mirrored entries are equal up to rounding of the fp64 FFT).  Must be
 * called before hfft_build_tensor / hfft_plan_set_buffers.  Errors: EINVAL, ESTATE.
 */
hfft_status hfft_plan_set_mirror(hfft_plan *plan, int on);

/*
 * Reciprocity storage of the bank, on top of the ky-mirror storage.
 * dz_i N_ij(X,Y) = dz_j N_ji(-X,-Y): in the real form of the coupling, S_ij := dz_i R_ij
 * satisfies S_ji = S_ij^T, so the bank keeps one 3 x 3 block per UNORDERED layer pair --
 * nz(nz+1)/2 instead of nz^2, half the bytes again -- the other orientation uses the
 * transpose (xz, yz negated) and H_i is multiplied by 1/dz_i at the end.
 *   on = 2 (default): automatic.  fp32 plans with 8 <= nz <= 64 whose bank is in the mirror
 *          storage use the block layout of the symmetric-matvec kernel (coupling_symv.cu):
 *          every block is read from HBM once and applied to both of its layer pairs inside
 *          one warp (info.mirror == 3), wherever that layout (nz padded to whole strips of
 *          four layers) streams at least 30 % fewer bytes than the mirror bank.
 *   on = 1: wherever the mirror storage is active: the block layout if fp32 and nz <= 64,
 *          else the p <= q bank read through a pair table by the streaming kernel
 *          (info.mirror == 2: saves memory, not time -- the second use of an entry is a
 *          second read).
 *   on = 0: never.
 * hfft_update_dz rewrites, in these modes too, only the stored blocks whose layer pair has the changed layer
 * between or at its two layers (the other blocks and the layout's zero padding are left alone).  Must be called before
 * hfft_build_tensor / hfft_plan_set_buffers.  Errors: EINVAL, ESTATE.
 */
hfft_status hfft_plan_set_recip(hfft_plan *plan, int on);

/* Fusion of the layer coupling into the y transforms (north_star (c); the F2^-1 [ sum_j3 ... ] F2 sandwich of Eq.24,
 * PAPER.md:177-178): stages S2, S3 and S4 run as ONE kernel in which a CTA takes the kx column of all 3 nz planes --
 * forward y transforms, coupling in shared memory, inverse y transforms -- so that M^ / H^ never reach global memory
 * and hfft_demag enqueues 3 kernels instead of 5 (info.fused == 1, info.launches_per_demag == 3).  It needs the plain
 * bank (no ky-mirror, reciprocity or deduplicated storage), two columns of 3 nz x 2ny complex plus the transform rows
 * within 222 KB of shared memory (the only bound on nz: e.g. nz <= 126 at ny = 16 and nz <= 15 at ny = 128 in fp32),
 * and no batched coupling.
 *   mode = 1 (default): automatic -- on the small grids (those too small for the wide-tile / mirror storage), which
 *          are bound by kernel launches; large grids keep the staged path with its smaller banks, which is faster
 *          there (measured: profiles/r02_fusion.md).
 *   mode = 2: wherever it fits (overrides the automatic ky-mirror / reciprocity storage, not hfft_plan_set_mirror(2)).
 *   mode = 0: never.
 * Must be called before hfft_build_tensor / hfft_plan_set_buffers.  Errors: EINVAL, ESTATE.
 */
hfft_status hfft_plan_set_fusion(hfft_plan *plan, int mode);

/*
 * Host-only helper (no device needed): the tensor classes hfft_plan_set_dedup works with.
 * dz: HOST array of nz thicknesses; cls_out: HOST array of nz*nz ints, cls_out[i*nz+j] = bank slot
 * of the pair (target i, source j); *n_classes = number of slots; *toeplitz = 1 when the thicknesses
 * are all equal (slot = |i-j|; the xz, yz entries of the pair carry a minus sign for i < j).
 * Errors: EINVAL (NULL pointers, nz < 1 or > HFFT_MAX_NZ, non-positive / non-finite dz).
 */
hfft_status hfft_tensor_classes(int nz, const double *dz, int *cls_out, int *n_classes, int *toeplitz);

/* Sizes the plan needs; valid after create and after every hfft_plan_set_* call (each of them may
 * change the storage and with it the sizes).  Errors: EINVAL. */
hfft_status hfft_plan_info(const hfft_plan *plan, hfft_info *info);

/* The two sizes a caller who brings its own buffers needs, = info.bank_bytes and
 * info.workspace_bytes.  0 for a NULL plan. */
size_t hfft_bank_bytes(const hfft_plan *plan);
size_t hfft_workspace_bytes(const hfft_plan *plan);

/*
 * Optional: hand the plan caller-owned DEVICE buffers (e.g. torch tensors) of
 * at least info.bank_bytes and info.workspace_bytes, 256-byte aligned.  The
 * caller keeps ownership and must keep them alive until hfft_destroy.  Without
 * this call hfft_build_tensor allocates both with cudaMalloc and hfft_destroy
 * frees them.  Errors: EINVAL, ESTATE (after build).
 */
hfft_status hfft_plan_set_buffers(hfft_plan *plan, void *bank, void *workspace);

/*
 * Timed setup.  On device: evaluates the generalized Newell
 * tensor N^{ab}_{ij}(p dx, q dy) for every layer pair and in-plane offset
 * (PAPER.md:52 Eq.5, :99 Eq.11 with the 4th term read as Y+dy [A1], :80-85
 * Eq.10, :123-132 Eq.16, other components by permutation PAPER.md:46) in
 * double-double arithmetic (the 64-term sums cancel catastrophically in plain
 * fp64, reading A16), places it on the 2nx x 2ny periodic grid (A10), takes its
 * in-plane FFT in fp64 (left factor of PAPER.md:177 Eq.24) and stores the real
 * (xx,yy,zz,xy) or imaginary (xz,yz) part in the plan precision.
 * Enqueues on `stream` (a cudaStream_t, may be NULL = default stream) and
 * synchronises that stream before returning (it frees its scratch memory).
 * Errors: ENOMEM, ECUDA.
 */
hfft_status hfft_build_tensor(hfft_plan *plan, void *stream);

/*
 * The hot path: one demagnetization-field evaluation (Eq.24).
 *   m   DEVICE pointer, [B][3][nz][ny][nx], plan precision, read only
 *   Ms  HOST pointer to nz doubles (per-layer saturation magnetisation, Eq.17
 *       PAPER.md:140, per-layer by reading A12), read during the call and passed
 *       by value to the kernels; NULL means 1.0 (m already holds M)
 *   h   DEVICE pointer, same shape and type as m, overwritten; units of Ms;
 *       the two arrays must not overlap, not even partially (EINVAL)
 * Only enqueues kernels on `stream`: no host synchronisation, no allocation,
 * safe to capture in a CUDA graph.  Consecutive calls on one plan share its spectra:
 * enqueue them on one stream (or order the streams yourself).  Errors: EINVAL,
 * ESTATE (tensor not built; evaluations of hfft_demag_host_async outstanding -- call
 * hfft_host_join first), ECUDA (launch failure).
 */
hfft_status hfft_demag(hfft_plan *plan, const void *m, const double *Ms, void *h, void *stream);

/*
 * Same evaluation with HOST buffers (pinned memory gives asynchronous copies):
 * copies m to a staging buffer of the plan, runs hfft_demag, copies h back, all on
 * `stream`.  Does not synchronise the stream.  The first host-path call of a plan
 * allocates the staging buffers (four arrays of the size of m; freed by
 * hfft_destroy).  Errors: as hfft_demag, ENOMEM.
 */
hfft_status hfft_demag_host(hfft_plan *plan, const void *m_host, const double *Ms, void *h_host,
                            void *stream);

/*
 * Pipelined form of hfft_demag_host for back-to-back evaluations (a time loop
 * feeding magnetisations from the host): the copy-in, the five kernels and the
 * copy-out run on three streams owned by the plan, with two staging slots, so
 * the PCIe transfers of evaluation n+1 / n-1 overlap the kernels of evaluation
 * n.  The call waits (on the device, not on the host) for everything enqueued on
 * `stream` before it, then returns at once; h_host is valid only after
 * hfft_host_join(plan, stream) followed by a synchronisation of `stream` (or of
 * an event recorded on it).  m_host must stay unchanged until then; pinned
 * memory is needed for the copies to be asynchronous.  Evaluations complete in
 * call order.  Not capturable in a CUDA graph.  Errors: as hfft_demag_host.
 */
hfft_status hfft_demag_host_async(hfft_plan *plan, const void *m_host, const double *Ms, void *h_host,
                                  void *stream);
/* Makes `stream` wait for every hfft_demag_host_async issued so far (no host blocking).  Until it is
 * called, hfft_demag and hfft_demag_host on this plan return ESTATE: they would use the spectra the
 * pipeline is still working on.  After it, issue them on `stream` (or on a stream ordered after it). */
hfft_status hfft_host_join(hfft_plan *plan, void *stream);

/*
 * Geometry update for layer-thickness optimisation (section 4
 * "Layer thickness optimization": the thickness of one layer is varied by a
 * Newton iteration and the tensor is rebuilt each time).
 * Sets dz[k] = dz_new and rebuilds ONLY the layer pairs whose tensor changes:
 * N_ij depends on (dz_i, dz_j, zeta_i - zeta_j) alone, so pairs with both layers
 * below k, or both above k, keep their entries; row i = k is rebuilt for all j,
 * rows i < k for j >= k, rows i > k for j <= k.  Same arithmetic as
 * hfft_build_tensor (double-double evaluation, fp64 FFT).  Enqueues on
 * `stream` and synchronises it before returning (frees its scratch memory).
 * Errors: EINVAL (k out of range, dz_new not positive / finite), ESTATE (tensor
 * not built), EUNSUPPORTED (deduplicated bank: use hfft_plan_set_dedup(plan, 0)),
 * ENOMEM, ECUDA (the plan then needs hfft_build_tensor again); ESTATE also while evaluations of
 * hfft_demag_host_async are outstanding (they read the bank on the plan's own streams): call hfft_host_join
 * first.  The same holds for a second hfft_build_tensor on a built plan.
 */
hfft_status hfft_update_dz(hfft_plan *plan, int k, double dz_new, void *stream);

/*
 * hfft_update_dz for callers that must not allocate device memory.
 *
 * Who this is for.  hfft_update_dz takes its setup scratch (info.setup_scratch_bytes) from
 * cudaMalloc and gives it back with cudaFree on EVERY call.  That is not possible for
 *   - a simulation code that has handed all of the GPU's memory to a pool of its own at start-up
 *     (a framework's caching allocator, a pre-sized arena): cudaMalloc then fails with "out of
 *     memory" although the program has room to spare;
 *   - a thickness-optimisation or real-time loop (PAPER.md:205-211 rebuilds the tensor at every
 *     Newton step) that cannot accept what cudaMalloc / cudaFree bring with them: a device-wide
 *     synchronisation, a driver lock, a run time that nobody bounds;
 *   - a host thread that works while another thread of the process records a CUDA graph in the
 *     global capture mode, where cudaMalloc is a forbidden call and breaks the recording.
 * This entry point does the same work -- same arguments, same kernels, same arithmetic, the bank
 * comes out bit for bit as from hfft_update_dz -- but its scratch is a fixed array that lives in
 * the library's device image.  It calls no cudaMalloc, no cudaFree and no library routine that
 * allocates device memory (on the host it uses a few small std::vector tables, as hfft_update_dz does).
 *
 * The limit.  The array has HFFT_STATIC_SCRATCH_BYTES = 32 MiB.  A plan whose
 * info.setup_scratch_bytes is larger is refused with HFFT_EUNSUPPORTED and a message that gives
 * both numbers; nothing has been touched then.  32 MiB holds e.g. 64 x 64 cells with up to 8
 * layers or 32 x 32 with up to 32 (the paper's 60 nm disc example, 64 x 64 x 5, needs 19 MB).
 * Larger plans use hfft_update_dz.
 *
 * What it costs.  Every GPU on which the CUDA runtime loads this part of the library holds the
 * 32 MiB from that moment -- at the latest the first call of this function on that GPU -- until the
 * process exits; hfft_destroy does not release it.
 *
 * First call on a device.  The first call made while a given device is current looks up the
 * array's address on that device (cudaGetSymbolAddress, which also makes the runtime load the
 * device image) and keeps it.  Make that first call at start-up, before any stream capture begins
 * anywhere in the process; later calls only read the stored address.
 *
 * Sharing.  All plans and all host threads of the process use the same array on a device, and it
 * keeps whatever the previous call left in it.  Nothing in the rebuild relies on old contents:
 * the one region that has to start at zero (the padded real-space tensor planes) is cleared on
 * the stream at the start of every call.  Two rebuilds running on the GPU at the same time would
 * overwrite each other's intermediate results and leave wrong banks without any error.  The
 * library keeps that from happening inside one process: the call holds a lock from its first
 * enqueue until it has synchronised `stream`, so a second caller waits.  Do not defeat it (for
 * instance by calling from a host callback of the same stream).
 *
 * Otherwise as hfft_update_dz: enqueues on `stream`, synchronises it before returning, commits
 * dz[k] only when the rebuild went through.  Errors: those of hfft_update_dz except ENOMEM, plus
 * EUNSUPPORTED for a plan beyond the limit.
 */
#define HFFT_STATIC_SCRATCH_BYTES (32u * 1024u * 1024u)
hfft_status hfft_update_dz_static(hfft_plan *plan, int k, double dz_new, void *stream);

/*
 * Fused reductions of the field.  With a non-NULL
 * `sums_device` (DEVICE pointer to B*3*nz*2 doubles, caller-owned, 8-byte
 * aligned) every following hfft_demag / hfft_demag_host zeroes that array and
 * its last kernel (S5) accumulates, for plane p = (b*3 + c)*nz + i,
 *     sums[2p]   = sum over the nx*ny cells of h_c(., ., i)          (<H_c> of layer i times nx*ny;
 *                  the quantity the paper's thickness optimisation drives to zero)
 *     sums[2p+1] = sum over the cells of m_c * h_c, m as passed to the call
 *                  (demagnetization energy: E = -(mu0/2) dx dy sum_i dz_i Ms_i sum_c sums[2p+1]
 *                  when Ms was passed per layer; Eq.1-2 define H as the cell average)
 * in fp64 (floating-point atomics: the summation order is not fixed).
 * NULL switches the reductions off (the default; no cost).  Errors: EINVAL.
 */
hfft_status hfft_plan_set_reduction(hfft_plan *plan, double *sums_device);

/*
 * Per-stage device timing.  With profiling on, hfft_demag brackets every stage
 * with CUDA events on `stream`.  hfft_profile_read synchronises on the last
 * event and returns, for each of the HFFT_NUM_STAGES stages, the SUM of elapsed
 * milliseconds over the calls since the last read, and the number of calls; it
 * then resets the sums.  At most 256 calls are kept between reads (further
 * calls return ESTATE).  Profiling makes hfft_demag unsuitable for graph capture.
 */
hfft_status hfft_profile_enable(hfft_plan *plan, int on);
hfft_status hfft_profile_read(hfft_plan *plan, double stage_ms[HFFT_NUM_STAGES], int *calls);

/*
 * Introspection for tests: copy one spectral bank plane N^_{ij}^{c}(k) to a
 * HOST array of n_k doubles, c in xx,yy,zz,xy,xz,yz = 0..5.  Element k =
 * kx * 2ny + ky, kx = 0..nx (Hermitian half spectrum along x), ky = 0..2ny-1.
 * The value is the real part for c < 4 and the imaginary part for c = 4, 5.
 * Synchronises the device.  Errors: EINVAL, ESTATE.
 */
hfft_status hfft_read_bank(const hfft_plan *plan, int i, int j, int c, double *out_host);

/* Release the plan and everything it owns.  NULL is allowed. */
hfft_status hfft_destroy(hfft_plan *plan);

/* Message of the last failing call on this plan ("" if none); plan may be NULL
 * to get the message of the last failing hfft_plan_create on this thread. */
const char *hfft_last_error(const hfft_plan *plan);

/* Library build identification, e.g. "hfft 0.4 sm_100a". */
const char *hfft_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HFFT_H */
