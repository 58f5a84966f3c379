/*
 * scwatter.h -- C ABI of libscw: B200-native (sm_100a) field evaluation for the coupled-wave
 * method of arXiv 2404.07293 ("sCWatter").  Citations are PAPER.md line numbers.
 *
 * The library evaluates the plane-wave-expanded electric field (discrete eq. 3)
 *
 *     E(r) = sum_j sum_m  c_j V[(comp,m), j] exp(i k s_m . (x,y)) G(gamma_j, zref_j, z)
 *
 * inside one sample layer (eq. 30/31/34, recomposed with eq. 10,
 * PAPER.md:119-124, 382) on rectilinear grids and at scattered points.
 *
 * CONVENTIONS
 *  - Every function returns an int32_t status (SCW_OK == 0).  Nothing throws, aborts or prints.
 *    All validation happens on the host BEFORE anything is enqueued; on error nothing is written.
 *    scw_last_error() returns a ctx-owned message for the last failing call.
 *  - Pointers are DEVICE pointers unless the comment says HOST.  Device pointers must be aligned
 *    to the complex element size (8 B for SCW_C64, 16 B for SCW_C128; 8 B for doubles).
 *  - Complex numbers are interleaved (re, im).  SCW_C64 = 2 x fp32, SCW_C128 = 2 x fp64.
 *  - Ownership: the caller owns every input, output and workspace buffer.  The library never
 *    allocates or frees device memory and keeps no caller pointer past the call, except the
 *    workspace registered with scw_set_workspace(), which it uses as scratch during calls.
 *  - Asynchrony: all work is enqueued on the ctx's CUDA stream; no call synchronises (the few that do say so).  Outputs
 *    are valid once the caller has synchronised that stream.  Descriptor structs are HOST memory
 *    and are copied by value during the call.  The device-buffer calls may be captured into a CUDA graph (stream
 *    capture) once the workspace has its final size; inputs and outputs of one call must not overlap.
 *  - One ctx per host thread.  There is no CPU fallback: scw_create fails with
 *    SCW_ERR_UNSUPPORTED on a device that is not compute capability 10.x.
 *
 * INDEXING (eq. 6): M = U*Vn spatial frequencies, m = (v + Vn/2)*U + (u + U/2),
 * u in [-floor(U/2), floor((U-1)/2)], s_m = lambda (u/X, v/Y).  Rows of V and P are comp*M + m with
 * comp = 0,1,2 for x,y,z (P = [P_x; P_y; P_z], eq. 28).
 * MODES (eq. 23/30): J columns, normally J = 4M.  A "+" mode
 * (dir = +1, gamma = +sqrt, Im gamma >= 0) is referenced at z_lo = z_{l-1}; a "-" mode
 * (dir = -1) at z_hi = z_l, so that every exponential decays inside [z_lo, z_hi].
 */
#ifndef SCWATTER_H
#define SCWATTER_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct scw_ctx scw_ctx;

enum {
    SCW_OK = 0,
    SCW_ERR_NULL = 1,        /* a required pointer is NULL */
    SCW_ERR_SHAPE = 2,       /* non-positive / inconsistent dimension, leading dimension too small */
    SCW_ERR_DTYPE = 3,       /* dtype is neither SCW_C64 nor SCW_C128 */
    SCW_ERR_ALIGN = 4,       /* device pointer not aligned to its element size */
    SCW_ERR_VALUE = 5,       /* lambda <= 0, X <= 0, Y <= 0, z_hi < z_lo, non-finite scalar */
    SCW_ERR_WORKSPACE = 6,   /* registered workspace too small; see scw_required_workspace() */
    SCW_ERR_CUDA = 7,        /* a CUDA runtime call failed; see scw_last_cuda_error() */
    SCW_ERR_UNSUPPORTED = 8  /* device is not sm_100-class, or an option value is unknown */
};

enum { SCW_C64 = 0, SCW_C128 = 1 };

/* Which kernels implement the two contractions (scw_set_option(ctx, SCW_OPT_PATH, v)). */
enum {
    SCW_OPT_PATH = 1,
    SCW_OPT_PROFILE = 2,  /* 0/1: record CUDA events around every kernel launch */
    SCW_OPT_CACHE = 3     /* 0/1: keep the twiddle tables F_x, F_y (step a-3; wavelength-free, eq. 6) in the workspace between
                             consecutive scw_sweep_wavelengths / scw_sweep_intensity calls.  While it is 1 the caller promises
                             that (i) the workspace is not written between those calls and (ii) the CONTENTS of x and y do not
                             change while their pointers, Nx, Ny, U, Vn, X, Y stay the same; call scw_invalidate_cache() after
                             changing coordinates in place.  Any other call on the ctx drops the cache.  Default 0. */
};
enum {
    SCW_PATH_AUTO = 0,    /* tcgen05 tensor-core kernels where shape/dtype allow, CUDA-core otherwise */
    SCW_PATH_SIMT = 1,    /* CUDA-core kernels only (fp32 FMA for C64, fp64 DFMA for C128) */
    SCW_PATH_TENSOR = 2   /* tensor-core kernels only; SCW_ERR_UNSUPPORTED if they cannot run */
};

/* ---------------------------------------------------------------- lifecycle */

/* Create a context bound to `device` and to `cuda_stream` (a cudaStream_t, may be 0 = legacy
 * default stream).  HOST: out.  Errors: NULL, CUDA, UNSUPPORTED. */
int32_t scw_create(scw_ctx** out, int32_t device, void* cuda_stream);
int32_t scw_destroy(scw_ctx* ctx);
int32_t scw_set_stream(scw_ctx* ctx, void* cuda_stream);
/* Register caller-owned device scratch (256-byte aligned).  May be (NULL, 0). */
int32_t scw_set_workspace(scw_ctx* ctx, void* dev_ptr, size_t bytes);
int32_t scw_set_option(scw_ctx* ctx, int32_t option, int64_t value);
int32_t scw_invalidate_cache(scw_ctx* ctx);
/* Message / raw cudaError_t / required workspace bytes of the last failing call on this ctx. */
const char* scw_last_error(const scw_ctx* ctx);
int32_t scw_last_cuda_error(const scw_ctx* ctx);
size_t scw_required_workspace(const scw_ctx* ctx);
/* Number of kernels this ctx has launched since creation (monotone counter). */
int64_t scw_launch_count(const scw_ctx* ctx);
/* Which kernels the last hot-path call on this ctx launched: bit k set = kernel class k (names: scw_profile_name(k)).  Lets a
 * caller see whether SCW_PATH_AUTO took the tensor-core kernels ("tc_assemble", "tc_synth", "dmma_*") or fell back to the
 * CUDA-core ones ("simt_*": complex64 beyond 80 frequencies per axis, V not 16-byte aligned, tiny problems, ...). */
uint64_t scw_last_kernels(const scw_ctx* ctx);
/* Library version: major*10000 + minor*100 + patch. */
int32_t scw_version(void);

/* Per-kernel device timers (only while SCW_OPT_PROFILE is 1): every launch is bracketed by CUDA events
 * on the ctx stream.  scw_profile_read synchronises on the recorded events and returns, for one kernel
 * class in [0, scw_profile_classes()), the accumulated device milliseconds and launch count since the
 * last scw_profile_reset (HOST out-pointers).  scw_profile_name returns a static string, NULL if out of range. */
int32_t scw_profile_classes(void);
const char* scw_profile_name(int32_t kernel_class);
int32_t scw_profile_read(scw_ctx* ctx, int32_t kernel_class, double* ms_total, int64_t* launches);
int32_t scw_profile_reset(scw_ctx* ctx);
/* Timeline of the last tensor-core assembly launch (always recorded, four globaltimer reads per CTA): for each of its
 * persistent CTAs the microseconds from the CTA's start to (0) its share of the mode weights written, (1) the weights of
 * all CTAs visible, (2) its span of V streamed, (3) exit after the fix-up.  us: HOST [max_ctas][4]; *n_ctas (HOST) = CTAs of
 * that launch (0 if none yet).  SYNCHRONISES the stream.  Errors: NULL, SHAPE (max_ctas too small), CUDA. */
int32_t scw_profile_assembly(scw_ctx* ctx, int32_t max_ctas, double* us, int32_t* n_ctas);
/* Device-clock timeline of the tensor-core sweep kernels (always recorded, one atomicMax per CTA): the last CTA of every
 * tcgen05 assembly / synthesis launch of a grouped sweep leaves the GPU's globaltimer (ns) at its exit in a ring of 128
 * slots inside the workspace.  Unlike the CUDA-event timers above this does not put anything between the kernels, so the
 * programmatic overlap of consecutive launches stays as in a plain run: the difference of two consecutive entries is the
 * time the later kernel added to the stream.  Returns the last min(max_n, 128, launches so far) launches, oldest first:
 * exit_ns[i] (HOST), kernel_class[i] (HOST; an index for scw_profile_name), *n (HOST).  Valid while the workspace of the
 * sweeps is untouched.  SYNCHRONISES the stream.  Errors: NULL, CUDA. */
int32_t scw_profile_timeline(scw_ctx* ctx, int32_t max_n, uint64_t* exit_ns, int32_t* kernel_class, int32_t* n);

/* ---------------------------------------------------------------- descriptors (HOST PODs) */

/* One layer at one wavelength. */
typedef struct {
    uint32_t struct_size;      /* = sizeof(scw_layer) */
    int32_t dtype;             /* SCW_C64 | SCW_C128: element type of V, c, P, E */
    int32_t U, Vn;             /* frequency grid (eq. 6) */
    double X, Y;               /* patch size, same unit as lambda (eq. 6) */
    double lambda;             /* vacuum wavelength, k = 2 pi / lambda (eq. 3) */
    double z_lo, z_hi;         /* z_{l-1}, z_l: the layer's interfaces (eq. 30) */
    int64_t J;                 /* number of modes (columns of V), normally 4*U*Vn (eq. 23) */
    const void* V;             /* [ldV x J] column-major complex<dtype>, rows comp*M+m (eq. 28, 34) */
    int64_t ldV;               /* >= 3*U*Vn; any value works, 64-byte aligned columns (ldV % 8 == 0 for C64) save ~3 % */
    const void* c;             /* [J] complex<dtype> coefficients alpha_j, NULL = ones (eq. 23) */
    const double* gamma;       /* [J] complex128 signed z-wavenumbers Gamma_jj (eq. 22-23) */
    const int8_t* dir;         /* [J] +1 / -1 reference face, NULL = derive from the sign of gamma */
} scw_layer;

enum { SCW_MODES_PLANEWAVE = 0, SCW_MODES_DENSE = 1 };

/* Mode table of the point path. */
typedef struct {
    uint32_t struct_size;      /* = sizeof(scw_modes) */
    int32_t kind;              /* SCW_MODES_PLANEWAVE | SCW_MODES_DENSE */
    /* SCW_MODES_PLANEWAVE: one plane wave per mode (eq. 3, eq. 9-10; any s_m) */
    int32_t dtype;             /* type of p and E */
    int64_t J;
    double lambda;
    const double* sx;          /* [J] direction cosines s_x = lambda u / X */
    const double* sy;          /* [J] */
    const double* gamma;       /* [J] complex128 s_z, signed */
    const double* zref;        /* [J] reference plane of each wave */
    const void* p;             /* [J x 3] complex<dtype> amplitudes, comp fastest */
    /* SCW_MODES_DENSE: the full eq. 34 of one layer at scattered points */
    scw_layer layer;
} scw_modes;

/* ---------------------------------------------------------------- the hot path */

/*
 * Spectral assembly (eq. 31 with the diag(alpha) factoring of PAPER.md:428-432):
 *   P[:, i] = V . ( c o g(z_i) ),  g_j(z) = G(gamma_j, zref_j, z) = exp(i k gamma_j (z - zref_j))  (eq. 7)
 * z: [Fz] doubles (device).  P: [ldP x Fz] column-major complex<dtype>, ldP >= 3*U*Vn.
 * z outside [z_lo, z_hi] is evaluated as-is.  Workspace: see scw_assemble_workspace().
 * Domain: every phase gamma_j (z - zref_j) / lambda is reduced to a fraction of a turn in fp64 before the trigonometric
 * functions, for both dtypes (SCW_C128: rint; SCW_C64: the low word of the 64-bit integer nearest to phase * 2^32, valid
 * for |phase| < 2^31 turns): any z of practical size gives the correctly reduced phase (the fp64 product itself carries
 * 2^-53 |phase| turns of rounding, which is what limits complex128 beyond ~1e5 turns).
 */
int32_t scw_assemble_spectra(scw_ctx* ctx, const scw_layer* layer, int64_t Fz, const double* z,
                             void* P, int64_t ldP);
int32_t scw_assemble_workspace(scw_ctx* ctx, const scw_layer* layer, int64_t Fz, size_t* bytes);

/*
 * Separable Fourier synthesis (eq. 10 on a rectilinear grid):
 *   E_comp(x_i, y_k, z_n) = sum_{u,v} P[comp*M + m(u,v), n] exp(i 2 pi (u x_i / X + v y_k / Y))
 * x: [Nx], y: [Ny] doubles (device).  E: complex<dtype>, element (comp, n, k, i) at offset
 * comp*strides[0] + n*strides[1] + k*strides[2] + i*strides[3] (in elements); strides == NULL
 * (HOST pointer) means planar [Fz][3][Ny][Nx], x fastest.
 */
int32_t scw_synthesize_grid(scw_ctx* ctx, int32_t dtype, int32_t U, int32_t Vn, double X, double Y,
                            int64_t Fz, const void* P, int64_t ldP,
                            int64_t Nx, const double* x, int64_t Ny, const double* y,
                            void* E, const int64_t* strides);
int32_t scw_synthesize_workspace(scw_ctx* ctx, int32_t dtype, int32_t U, int32_t Vn, int64_t Fz,
                                 int64_t Nx, int64_t Ny, size_t* bytes);

/*
 * Scattered points (eq. 3 / eq. 9-10 for SCW_MODES_PLANEWAVE, eq. 34 for SCW_MODES_DENSE).
 * r: [N x 3] doubles (x,y,z per point).  E: [N x 3] complex<dtype>, comp fastest.
 * Domain: any finite coordinates.  The phase k s . r is range-reduced in fp64: SCW_C128 reduces every term with rint;
 * SCW_C64 takes phases relative to the first point r_0 of the call (the per-wave phase at r_0 is reduced with rint)
 * and sums the three fp64 products onto the constant 1.5 * 2^20, exact while the phase relative to r_0 stays below
 * 2^19 turns; a block of 512 points that holds a point beyond that bound (|s|_max |r - r_0| / lambda >= 524 000)
 * reduces every term with rint as well, at ~1.3x the time for that block.  The amplitude exponent
 * -k Im(gamma) (z - zref) is evaluated in fp32 relative to z_0: its error grows as 2^-24 k |Im gamma| |z - z_0|.
 */
int32_t scw_eval_points(scw_ctx* ctx, const scw_modes* modes, int64_t N, const double* r, void* E);
int32_t scw_points_workspace(scw_ctx* ctx, const scw_modes* modes, int64_t N, size_t* bytes);

/*
 * scw_eval_points for callers that cannot hand the library any scratch memory.
 *
 * Who this is for: code that runs where device memory can no longer be obtained -- a plug-in called from inside a host
 * application whose memory pool already owns the whole GPU, a real-time loop that has promised not to touch the allocator
 * after start-up (cudaMalloc takes a process-wide lock and may synchronise the device), or an out-of-memory handler that
 * still wants one last field evaluation.  Such a caller cannot cudaMalloc a workspace for
 * scw_set_workspace, and scw_eval_points needs one for complex64 plane-wave tables (it tabulates the J waves there
 * before summing them).
 *
 * This call needs none and allocates nothing: no cudaMalloc / cudaFree, no event or stream creation, no workspace.
 * Its table lives in a fixed array compiled into libscw.so (SCW_POINTS_NOALLOC_MAX_J entries of 96 bytes plus a
 * 256-byte header, 768.25 KiB); every GPU that loads the library carries that array until the process exits, whether
 * or not this function is ever called.  Only the SCW_MODES_PLANEWAVE kind is served (the dense kind needs scratch that
 * grows with M * N).  modes, N, r, E: exactly as scw_eval_points; inputs and outputs stay the caller's.  The registered
 * workspace, if any, is neither needed nor touched.  The arithmetic is that of scw_eval_points (same kernels, same
 * domain notes): for equal inputs the two calls return equal fields.
 *
 * Limit: J <= SCW_POINTS_NOALLOC_MAX_J for SCW_C64; a larger table is refused with SCW_ERR_SHAPE before anything is
 * enqueued (scw_last_error names the limit).  SCW_C128 tables use no scratch and are accepted at any J.
 *
 * First call on a device: it looks up where that GPU keeps the array (once per device per process, under a lock; this
 * may make the CUDA runtime load the library's kernels on that GPU).  Make that first call during start-up, before any
 * stream capture begins; later calls only enqueue one 24-byte memset and two kernels on the ctx stream.  A
 * cudaDeviceReset() invalidates the looked-up address: do not reset a device this function has been used on.
 *
 * Sharing: there is ONE array per GPU, shared by every ctx, stream and host thread of the process, and it keeps what the
 * last call left in it.  The call rewrites what it reads (the header is cleared, the J table entries are rebuilt) in
 * stream order, so back-to-back calls on one stream are safe.  Two calls that can overlap on the same GPU -- different
 * streams, different ctxs, different threads -- race on the table and return garbage: order them yourself (one stream,
 * or an event between them).
 * Errors: NULL, SHAPE (N < 0, J <= 0, J above the limit, wrong struct_size), DTYPE, ALIGN, VALUE,
 * UNSUPPORTED (SCW_MODES_DENSE), CUDA (address look-up or launch failed; see scw_last_cuda_error).
 */
#define SCW_POINTS_NOALLOC_MAX_J 8192
int32_t scw_eval_points_noalloc(scw_ctx* ctx, const scw_modes* modes, int64_t N, const double* r, void* E);

/*
 * Batched grid evaluation: assembly + synthesis for every (wavelength, layer) instance in one
 * call (spectroscopy sweep).  All instances share U, Vn, X, Y, dtype and the
 * x/y grid (the twiddles are wavelength-free: k s_m . r = 2 pi (u x/X + v y/Y), eq. 6).  J and Fz may differ between
 * instances: consecutive instances with the same J and Fz (up to 64) form a run that is evaluated by ONE assembly launch and
 * ONE synthesis launch; an instance the tensor-core kernels cannot take (see scw_last_kernels) puts the whole call on the
 * per-instance path.
 * inst: HOST [n_inst].  Fz: HOST [n_inst].  z: HOST array of device pointers.  E: HOST array of
 * device pointers, each laid out by `strides` as in scw_synthesize_grid.
 */
int32_t scw_sweep_wavelengths(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst,
                              const int64_t* Fz, const double* const* z,
                              int64_t Nx, const double* x, int64_t Ny, const double* y,
                              void* const* E, const int64_t* strides);
int32_t scw_sweep_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz,
                            int64_t Nx, int64_t Ny, size_t* bytes);

/*
 * Calibrate the work split of the tensor-core assembly (step a-2) for this device and this workload: its persistent CTAs
 * (one per SM) each stream a contiguous span of V, and the SMs do not all reach the same HBM rate (the same groups of SMs
 * are slower in every run; by how much depends on what else the memory system is doing when the kernel starts).  Runs the
 * given sweep -- arguments and outputs exactly as scw_sweep_wavelengths -- `reps` + 1 times per round for nine rounds,
 * measures every CTA of its assembly launch, moves the spans half way towards the measured relative rates after each round
 * and keeps, for all later calls on this ctx, the split whose assembly finished earliest (the equal split if none beat it;
 * results change only in summation order).  SYNCHRONISES the stream.  A sweep that does not take the tensor-core
 * assembly is accepted and leaves the equal split.  reps in [1, 64].  Errors: those of scw_sweep_wavelengths, VALUE (reps).
 */
int32_t scw_calibrate(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, const double* const* z,
                      int64_t Nx, const double* x, int64_t Ny, const double* y, void* const* E, const int64_t* strides,
                      int32_t reps);

/*
 * Same as scw_sweep_wavelengths with every array in HOST memory (V, c, gamma, dir, z[i], x, y, E[i];
 * pinned memory required for overlap): inputs are staged host->device into the workspace, evaluated, and E is
 * copied device->host.  Two staging buffers each way and two internal copy streams pipeline the instances (the upload of
 * instance i+1 and the download of instance i-1 run beside the kernels of instance i); the pipeline is forked from and
 * joined back into the ctx stream with events, so results are complete in ctx-stream order.  E[i] is planar [Fz][3][Ny][Nx].  h2d_bytes / d2h_bytes
 * (HOST, may be NULL) receive the bytes copied in each direction.
 */
int32_t scw_sweep_wavelengths_host(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst,
                                   const int64_t* Fz, const double* const* z,
                                   int64_t Nx, const double* x, int64_t Ny, const double* y,
                                   void* const* E, int64_t* h2d_bytes, int64_t* d2h_bytes);
int32_t scw_sweep_host_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst,
                                 const int64_t* Fz, int64_t Nx, int64_t Ny, size_t* bytes);

/* ---------------------------------------------------------------- exterior field
 *
 * Field in the homogeneous half-spaces above (z <= z_0) and below (z >= z_L) the sample, eq. 9:
 *   above:  p(s_m, z) = p_inc_m  G[ s_z(n), z_inc,  z]  +  p_face_m G[-s_z(n), z_face, z]     (incident + reflected)
 *   below:  p(s_m, z) = p_face_m G[ s_z(n), z_face, z]                                         (transmitted)
 * with s_z(n) = sqrt(n^2 - |s_m|^2), Im >= 0 (eq. 2), s_m = lambda (u/X, v/Y) (eq. 6), G of eq. 7, followed by
 * eq. 10, E(r, z) = sum_m p(s_m, z) exp(i k s_m . r).  The reflected wave travels toward -z: its z-wavenumber is
 * -s_z(n), so that it decays away from the interface it is referenced at (reading c-17).
 * Amplitudes are [M x 3] complex<dtype>, component fastest, m as in eq. 6's index map (u fastest).
 */
enum { SCW_SIDE_ABOVE = 0, SCW_SIDE_BELOW = 1 };
typedef struct {
    uint32_t struct_size;      /* = sizeof(scw_exterior) */
    int32_t dtype;             /* SCW_C64 | SCW_C128: element type of the amplitudes, P and E */
    int32_t side;              /* SCW_SIDE_ABOVE | SCW_SIDE_BELOW */
    int32_t U, Vn;             /* frequency grid (eq. 6) */
    double X, Y;               /* patch size */
    double lambda;             /* vacuum wavelength */
    double n_re, n_im;         /* refractive index of the half-space (real above, complex below) */
    double z_face;             /* z_0 (above) or z_L (below): reference plane of p_face */
    double z_inc;              /* z-bar: reference plane of the incident wave (above only) */
    const void* p_face;        /* [M x 3] reflected (above) / transmitted (below) amplitudes, device */
    const void* p_inc;         /* [M x 3] incident amplitudes (above only), device; NULL = no incident wave */
} scw_exterior;

/* eq. 9 on Fz planes: P[comp*M + m, i] = p_comp(s_m, z_i), column-major [ldP x Fz], ldP >= 3*U*Vn; feed P to
 * scw_synthesize_grid for eq. 10 on a rectilinear grid.  z: [Fz] doubles (device), evaluated as-is on either side.
 * No workspace.  Errors: NULL, SHAPE, DTYPE, ALIGN, VALUE, CUDA. */
int32_t scw_exterior_spectra(scw_ctx* ctx, const scw_exterior* ext, int64_t Fz, const double* z, void* P, int64_t ldP);

/* eq. 9 followed by eq. 10 on a rectilinear grid in ONE call: E as in scw_synthesize_grid (strides, planar default).  For
 * SCW_C64 with at most 80 frequencies per axis eq. 9 is evaluated straight into the synthesis kernel's operand (P is never
 * written) and the twiddle tables are kept under SCW_OPT_CACHE like a sweep's; otherwise it is scw_exterior_spectra into
 * the workspace + the synthesis.  Errors: as scw_exterior_spectra and scw_synthesize_grid, WORKSPACE. */
int32_t scw_exterior_grid(scw_ctx* ctx, const scw_exterior* ext, int64_t Fz, const double* z,
                          int64_t Nx, const double* x, int64_t Ny, const double* y, void* E, const int64_t* strides);
int32_t scw_exterior_grid_workspace(scw_ctx* ctx, const scw_exterior* ext, int64_t Fz, int64_t Nx, int64_t Ny, size_t* bytes);

/* eq. 9-10 at scattered points: the M (below) or 2M (above) plane waves are tabulated in the workspace and summed by
 * the direct plane-wave kernels of scw_eval_points.  r: [N x 3] doubles, E: [N x 3] complex<dtype>, comp fastest. */
int32_t scw_exterior_points(scw_ctx* ctx, const scw_exterior* ext, int64_t N, const double* r, void* E);
int32_t scw_exterior_points_workspace(scw_ctx* ctx, const scw_exterior* ext, int64_t N, size_t* bytes);

/* ---------------------------------------------------------------- detector reductions
 *
 * scw_sweep_wavelengths followed by what a detector records instead of the complex field (PAPER.md:422, 520-524, 544-546,
 * 554; reading c-18), with the field never written: on the tensor-core path the reductions run in the synthesis
 * epilogue.
 *   I(x, y, z)  = sum_comp |E_comp(x, y, z)|^2                    intensity per sample (4 bytes leave the SM instead of 24)
 *   S(z)        = sum_{(i, k) in window} I(x_i, y_k, z)           intensity collected by a detector window of the plane
 *                                                                  (plain sum over grid samples; multiply by dx dy for an area integral)
 *   A           = -log10(S / S_0)                                  absorbance against a reference sweep (scw_absorbance)
 * I: HOST array of device pointers, real (float for SCW_C64, double for SCW_C128), element (n, k, i) at
 * n*strides[0] + k*strides[1] + i*strides[2] elements; strides == NULL means [Fz][Ny][Nx], x fastest.  I == NULL: no per-
 * sample output.  S: HOST array of device pointers, real [Fz[i]] per instance; S == NULL: no window sums.  At least one of
 * I, S.  window: HOST, grid-index box [ix0, ix1) x [iy0, iy1) of the (x, y) grid; NULL = the whole plane.
 * Errors: those of scw_sweep_wavelengths; SHAPE for an empty window or one outside the grid.
 */
typedef struct { int64_t ix0, ix1, iy0, iy1; } scw_window;
int32_t scw_sweep_detector(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst,
                           const int64_t* Fz, const double* const* z,
                           int64_t Nx, const double* x, int64_t Ny, const double* y,
                           void* const* I, const int64_t* strides, const scw_window* window, void* const* S);
int32_t scw_sweep_detector_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz,
                                     int64_t Nx, int64_t Ny, size_t* bytes);
/* scw_sweep_detector with I only (whole plane, no window sums). */
int32_t scw_sweep_intensity(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst,
                            const int64_t* Fz, const double* const* z,
                            int64_t Nx, const double* x, int64_t Ny, const double* y,
                            void* const* I, const int64_t* strides);
int32_t scw_sweep_intensity_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz,
                                      int64_t Nx, int64_t Ny, size_t* bytes);
/*
 * Absorbance spectrum (Fig. 6): A[i] = -log10(S[i] / S0[i]) for n detector readings S (e.g. one per
 * wavelength of a sweep) against the readings S0 of a reference sweep, and / or the absorbance of the whole band,
 * band[0] = -log10( sum_i w_i S_i / sum_i w_i S0_i ) with spectral weights w (NULL = ones).  dtype SCW_C64: float arrays,
 * SCW_C128: double.  All device pointers; A or band may be NULL (not both).  Errors: NULL, DTYPE, SHAPE, ALIGN, CUDA.
 */
int32_t scw_absorbance(scw_ctx* ctx, int32_t dtype, int64_t n, const void* S, const void* S0, const void* w, void* A,
                       void* band);

/* ---------------------------------------------------------------- V builder
 *
 * The step upstream of the field evaluation: from the eigenvector matrix Q of a layer's property matrix (eq. 19-23,
 * PAPER.md:184-246; rows [P_x; P_y; B_x; B_y] in blocks of M, one column per mode) to the matrix V = T Q [diag(alpha)]
 * of scw_layer.  The P_x, P_y rows are copied; the P_z rows follow from eq. 33:
 *     [P_z]_m = + sum_{m'} psi_{m'} { [s_y]_{m-m'} [b_x]_{m-m'} - [s_x]_{m-m'} [b_y]_{m-m'} },   s_m = lambda (u/X, v/Y),
 * the 2-D circular convolution (per-axis wrap of the frequency difference onto the grid of eq. 6; the block-circulant
 * form of the matrix printed as eq. 21) of q = s_y o B_x - s_x o B_y with the Fourier-series coefficients psi of 1/n^2,
 * 1/n^2(r) = sum_m psi_m exp(ik s_m . r) (eq. 12 with that normalisation: a homogeneous layer has psi = delta_{(0,0)} / n^2).
 * The sign is + : with B = s x P (eq. 15, and eq. 21's D) only this sign gives s . p = 0 (eq. 14); the minus printed in
 * eq. 33 comes from the curl written with the opposite sign at PAPER.md:344 (readings c-19..c-21).
 * Runs as an M x M by M x J complex GEMM on the tensor cores.  V: [ldV x J] column-major complex<dtype>, ldV >= 3M.
 * Errors: NULL, SHAPE, DTYPE, ALIGN, VALUE, WORKSPACE, CUDA.
 */
typedef struct {
    uint32_t struct_size;      /* = sizeof(scw_vbuild) */
    int32_t dtype;             /* SCW_C64 | SCW_C128: element type of Q, psi, alpha, V */
    int32_t U, Vn;             /* frequency grid (eq. 6) */
    double X, Y;               /* patch size */
    double lambda;             /* vacuum wavelength */
    int64_t J;                 /* columns of Q (modes), normally 4*U*Vn */
    const void* Q;             /* [ldQ x J] column-major complex<dtype>, rows [P_x; P_y; B_x; B_y] (eq. 19-20) */
    int64_t ldQ;               /* >= 4*U*Vn */
    const void* psi;           /* [M] complex<dtype>, index m of eq. 6 */
    const void* alpha;         /* [J] complex<dtype> or NULL: fold diag(alpha) into V (then pass c = NULL to the evaluation) */
} scw_vbuild;
int32_t scw_build_V(scw_ctx* ctx, const scw_vbuild* vb, void* V, int64_t ldV);
int32_t scw_build_V_workspace(scw_ctx* ctx, const scw_vbuild* vb, size_t* bytes);

/* ---------------------------------------------------------------- alpha propagation
 *
 * The coefficient vectors alpha^(l) of every layer of a stack from the field vector at its top interface, by the
 * boundary conditions of PAPER.md:252-296 (eq. 24-26; interface matrices as de-garbled in DESIGN.md reading c-7):
 *     alpha^(1) = Q'_1^-1 r_0                         r_0 = Gbar Rbar + Rhat, the field [P_x; P_y; B_x; B_y] at z_0   (eq. 24)
 *     alpha^(l) = Q'_l^-1 Q`_{l-1} alpha^(l-1)                                                                      (eq. 25)
 *     r_L       = Q`_L alpha^(L)                      the field at the bottom interface z_L                          (eq. 26)
 *     Q'_l = Qcheck^(l) + Qhat^(l) G(Gamma^(l), z_l, z_{l-1}),   Q`_l = Qcheck^(l) G(Gamma^(l), z_{l-1}, z_l) + Qhat^(l)
 * with Qcheck / Qhat the "+" / "-" columns of the eigenvector matrix Q^(l) (dir as in scw_layer) and G of eq. 7.  Per
 * layer: one dense complex LU (partial pivoting, blocked, trailing updates on the FP64 tensor cores) and two triangular
 * solves; all arithmetic in fp64, SCW_C64 inputs and outputs are widened / rounded at the boundary.
 * r0, rL: [n] complex<dtype> (device); alpha: HOST array of n_layers device pointers [n]; rL may be NULL.
 * Pivoting: the pivot of column k is the entry of largest |re| + |im| at or below the diagonal (LAPACK's izamax measure);
 * among equal candidates the one in the smallest row wins, so the factorisation does not depend on the launch geometry.
 * A singular Q^(l), or one that holds NaN, gives non-finite alpha (no error is raised: nothing is read back); the ctx
 * and the device stay usable.
 * Errors: NULL, SHAPE, DTYPE, ALIGN, VALUE, WORKSPACE, UNSUPPORTED (n > 128 x #SMs or > 25 600), CUDA.
 */
typedef struct {
    uint32_t struct_size;          /* = sizeof(scw_stack) */
    int32_t dtype;                 /* SCW_C64 | SCW_C128: element type of Q, r0, alpha, rL */
    int32_t n_layers;              /* L */
    int64_t n;                     /* order of Q: 4M */
    double lambda;                 /* vacuum wavelength */
    const double* z_if;            /* HOST [L + 1]: interfaces z_0 <= ... <= z_L */
    const void* const* Q;          /* HOST [L] device pointers: Q^(l), [ldQ x n] column-major complex<dtype> */
    int64_t ldQ;                   /* >= n */
    const double* const* gamma;    /* HOST [L] device pointers: Gamma^(l), [n] complex128 signed (as scw_layer.gamma) */
    const int8_t* const* dir;      /* HOST [L] device pointers [n] (+1 / -1), or NULL: derive from the sign of gamma */
} scw_stack;
int32_t scw_propagate_alpha(scw_ctx* ctx, const scw_stack* st, const void* r0, void* const* alpha, void* rL);
int32_t scw_propagate_alpha_workspace(scw_ctx* ctx, const scw_stack* st, size_t* bytes);

/* ---------------------------------------------------------------- roofline denominators (measurement helper)
 *
 * Runs a small microbenchmark of one hardware unit on the ctx stream and returns its measured rate (best of `reps`
 * launches, CUDA events).  Unlike every other call this one SYNCHRONISES the stream.  buf: device scratch of `bytes`
 * bytes (contents destroyed); the HBM units stream through all of it -- pass >= 1 GiB so that it exceeds the L2;
 * the arithmetic units need 256 bytes.  value (HOST): TFLOP/s for FP64_DMMA (mma.sync.m8n8k4.f64, the complex128
 * contractions) and FP32_FMA, Gop/s for MUFU (ex2.approx: the pipe of the point path's sin / cos / ex2) and MUFU_MIX (one
 * sin.approx, one cos.approx and one ex2.approx per term, the point kernel's own mix: 3 ops per term), GB/s for
 * HBM_READ (16-byte loads), HBM_WRITE (16-byte st.global) and HBM_WRITE_TMA (16 KB cp.async.bulk shared -> global).
 * Errors: NULL, VALUE (unknown unit, reps < 1), CUDA.
 */
enum { SCW_PEAK_FP64_DMMA = 0, SCW_PEAK_FP32_FMA = 1, SCW_PEAK_MUFU = 2, SCW_PEAK_HBM_READ = 3, SCW_PEAK_HBM_WRITE = 4,
       SCW_PEAK_HBM_WRITE_TMA = 5, SCW_PEAK_MUFU_MIX = 6 };
int32_t scw_measure_peak(scw_ctx* ctx, int32_t which, void* buf, size_t bytes, int32_t reps, double* value);

#ifdef __cplusplus
}
#endif
#endif /* SCWATTER_H */
