// Internal declarations shared by the translation units of libscw (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <vector>
#include "scwatter.h"

namespace scw {
// Kernel classes for launch accounting and the optional per-kernel CUDA-event timers.
enum KernelClass {
    KC_WEIGHTS = 0, KC_TWIDDLES, KC_ASSEMBLE, KC_REDUCE, KC_SYNTH_A, KC_SYNTH_B, KC_POINTS_TABLE, KC_POINTS,
    KC_POINT_SYNTH, KC_MISC, KC_ASSEMBLE_TC, KC_SYNTH_TC, KC_SYNTH_IMG, KC_ASSEMBLE_DMMA, KC_SYNTH_A_DMMA, KC_SYNTH_B_DMMA, KC_EXTERIOR, KC_VBUILD_PREP, KC_ALPHA, KC_ALPHA_LU, KC_ALPHA_PANEL, KC_COUNT
};
struct ProfRec { cudaEvent_t a, b; int kc; bool owns_a; };
}  // namespace scw

struct scw_ctx {
    int device = 0;
    int sm_count = 148;
    cudaStream_t stream = nullptr;
    // host-buffer sweep only: copy streams and events of the double-buffered staging pipeline (forked from and joined
    // back into `stream`, so the caller still sees plain stream order)
    cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
    cudaEvent_t ev_start = nullptr, ev_in[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr},
                ev_out[2] = {nullptr, nullptr};
    void* ws = nullptr;
    size_t ws_bytes = 0;
    int64_t path = SCW_PATH_AUTO;
    int64_t launches = 0;
    uint64_t last_classes = 0;      // bit kc set: the last API call launched a kernel of class kc (scw_last_kernels)
    int32_t cuda_err = 0;
    size_t required_ws = 0;
    char msg[256] = {0};
    bool profile = false;
    bool tc_error = false;          // a tensor map could not be encoded (reported by the entry point)
    // stream-K split of the tcgen05 assembly: relative rate of every persistent CTA (scw_calibrate), empty = equal spans
    std::vector<double> split_w;
    int last_asm_G = 0;             // the last assembly launch: grid, spans, where its per-CTA nanoseconds are (device)
    int64_t last_asm_span0[161] = {0};
    const unsigned long long* last_asm_ns = nullptr;
    // twiddle cache (SCW_OPT_CACHE): key of the twiddle images held in the workspace, and the control block known clean
    bool cache_on = false;
    struct TwKey { const void *x = nullptr, *y = nullptr, *where = nullptr; int64_t Nx = 0, Ny = 0; int U = 0, Vn = 0, dtype = -1;
                   double X = 0, Y = 0; bool tc = false; } tw_key;
    bool tw_valid = false;
    const void* clean_ctl = nullptr;
    size_t clean_ints = 0;
    // spectrum-image buffer whose padding is known to hold zeros (same promise): location, frequency grid, planes
    const void* clean_img = nullptr;
    int clean_img_U = 0, clean_img_Vn = 0;
    int64_t clean_img_planes = 0;
    // device-clock timeline of the tensor-core sweep kernels (scw_profile_timeline): every such launch leaves the
    // globaltimer value of its last CTA's exit in slot (tl_seq % TL_RING) of a ring that lives in the assembly's control
    // block (caller's workspace); tl_ring is only valid inside the API call that set it (reset by check_ctx)
    unsigned long long* tl_ring = nullptr;
    const unsigned long long* tl_last_ring = nullptr;   // where the ring of the last sweep is (read back on request)
    int64_t tl_seq = 0;
    int tl_class[128] = {0};
    cudaEvent_t prof_last = nullptr;   // profiling: end event of the previous kernel of this API call
    std::vector<scw::ProfRec> recs;
    double prof_ms[scw::KC_COUNT] = {0};
    int64_t prof_n[scw::KC_COUNT] = {0};
};

namespace scw {

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

// Timeline ring (see scw_ctx::tl_ring): the slot the next launch of class kc stamps its exit time into, NULL if no ring.
constexpr int TL_RING = 128;
static_assert(sizeof(((scw_ctx*)nullptr)->tl_class) / sizeof(int) == TL_RING, "scw_ctx::tl_class holds one class per ring slot");
inline unsigned long long* tl_next(scw_ctx* ctx, int kc)
{
    if (!ctx->tl_ring) return nullptr;
    const int slot = (int)(ctx->tl_seq % TL_RING);
    ctx->tl_class[slot] = kc;
    ctx->tl_seq++;
    return ctx->tl_ring + slot;
}

// Brackets one kernel launch: counts it and, when profiling is on, times it with CUDA events on the ctx stream (read
// back by scw_profile_read).  A kernel's interval runs from the end event of the previous kernel of the same API call
// (a fresh start event for the first one) to its own end event: one event between consecutive kernels, and the
// intervals of a call add up to the call's span on the device, dependency gaps included.
struct KernelScope {
    scw_ctx* ctx;
    ProfRec rec;
    bool on;
    KernelScope(scw_ctx* c, int kc) : ctx(c), on(c->profile)
    {
        ctx->launches++;
        ctx->last_classes |= 1ull << kc;
        rec.kc = kc;
        if (on) {
            rec.owns_a = ctx->prof_last == nullptr;
            if (rec.owns_a) {
                cudaEventCreate(&rec.a);
                cudaEventRecord(rec.a, ctx->stream);
            } else {
                rec.a = ctx->prof_last;
            }
            cudaEventCreate(&rec.b);
        }
    }
    ~KernelScope()
    {
        if (on) {
            cudaEventRecord(rec.b, ctx->stream);
            ctx->prof_last = rec.b;
            ctx->recs.push_back(rec);
        }
    }
};

// Launch with programmatic stream serialization (PDL): the kernel's prologue -- everything before its pdl_wait() -- may
// overlap the tail of the previous kernel of the stream.
template <typename P>
inline void launch_pdl(void (*kernel)(P), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, const P& params)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kernel, params);
}

// Bump allocator over the caller's workspace.
struct Carver {
    char* base;
    size_t off = 0;
    explicit Carver(void* p) : base(static_cast<char*>(p)) {}
    void* take(size_t bytes) {
        void* p = base ? base + off : nullptr;
        off += align_up(bytes);
        return p;
    }
};

// ---- kernels_simt.cu ----------------------------------------------------------------------
// W[j*Fz + i] = c_j * exp(i 2 pi gamma_j (z_i - zref_j) / lambda)  (eq. 7, 30)
void launch_mode_weights(scw_ctx* ctx, int dtype, int64_t J, int64_t Fz, double lambda, double z_lo,
                         double z_hi, const void* c, const double* gamma, const int8_t* dir,
                         const double* z, void* W);
// Ft[f*N + i] = exp(i 2 pi (f - nfreq/2) coord_i / period)  (eq. 6, 10) -- frequency-major table
void launch_twiddles(scw_ctx* ctx, int dtype, int nfreq, int64_t N, const double* coord, double period,
                     void* Ft);
// P[r + i*ldP] = sum_j V[r + j*ldV] W[j*Fz + i]   (eq. 31)
size_t simt_assemble_scratch(int dtype, int64_t R, int64_t J, int64_t Fz, int sm_count);
void launch_simt_assemble(scw_ctx* ctx, int dtype, int64_t R, int64_t J, int64_t Fz, const void* V,
                          int64_t ldV, const void* W, void* P, int64_t ldP, void* scratch);
// Two-pass separable synthesis (eq. 10): T = P_comp Fy^T, E = Fx T.
size_t simt_synth_scratch(int dtype, int U, int64_t Fz, int64_t Ny);
void launch_simt_synth(scw_ctx* ctx, int dtype, int U, int Vn, int64_t Fz, const void* P, int64_t ldP,
                       int64_t Nx, const void* FxT, int64_t Ny, const void* FyT, void* E,
                       const int64_t strides[4], void* scratch);

// I[n][k][i] = sum_comp |E[n][comp][k][i]|^2, E planar, I at n*s3[0] + k*s3[1] + i*s3[2]
void launch_intensity(scw_ctx* ctx, int dtype, int64_t Fz, int64_t Ny, int64_t Nx, const void* E, void* I,
                      const int64_t s3[3]);
// S[n] = sum over the window (ix0, ix1, iy0, iy1; grid indices, half-open) and the components of |E[n][comp][k][i]|^2, E planar
void launch_window_sum(scw_ctx* ctx, int dtype, int64_t Fz, int64_t Ny, int64_t Nx, const void* E, const int64_t win[4], void* S);
// A[i] = -log10(S[i] / S0[i]); band (may be NULL): -log10(sum w S / sum w S0) over the n entries (w NULL = ones)
void launch_absorbance(scw_ctx* ctx, int dtype, int64_t n, const void* S, const void* S0, const void* w, void* A, void* band);

// ---- scw_tc_assemble.cu: tcgen05 BF16x3 spectral assembly (complex64) ----------------------------
bool tc_assemble_supported(int dtype, int64_t R, int64_t J, int64_t Fz, const void* V, int64_t ldV);
int tc_assemble_max_group();
size_t tc_assemble_scratch(const scw_ctx* ctx, int64_t R, int64_t J, int64_t Fz, int n_inst);
// Where the control block (arrival counters, must be zero at launch) of an assembly over `scratch` lies.
void tc_assemble_ctl(const scw_ctx* ctx, int64_t R, int64_t J, int64_t Fz, int n_inst, void* scratch, int** ctl, size_t* n_ints);
// What the assembly kernel's fix-up writes once a tile is complete.
enum { TC_FIX_P = 0, TC_FIX_IMAGES = 1, TC_FIX_NONE = 2 };
struct TcFixup {
    int mode;
    int64_t R;                  // rows of P (3M), filled in by the launcher
    // TC_FIX_P: instance i -> P + i*inst_stride, column-major [ldP x Fz] complex64
    float2* P;
    int64_t ldP, inst_stride;
    // TC_FIX_IMAGES: spectrum images of k_tc_synth (scw_tc_synth.cu): image ((inst*Fz + n)*3 + comp, uc, vc), hi | lo,
    // N1 rows x K1p, K-major core-matrix layout; chunks of Uc x Vc frequencies
    uint8_t* img;
    int U, Vn, Uc, Vc, nuc, nvc, K1p, N1;
    int skip_zero;              // the padding of the images already holds zeros (left by the previous launch)
};
// weights (a-1) + P = V W (a-2) + fix-up, n_inst <= tc_assemble_max_group() instances with equal U, Vn, J, Fz in ONE launch;
// sched/n_sched: plane counters of the synthesis that follows (zeroed by the kernel), may be NULL.
void launch_tc_assemble_group(scw_ctx* ctx, int n_inst, const scw_layer* inst, int64_t Fz, const double* const* z,
                              const TcFixup& fix, int* sched, int n_sched, void* scratch, bool ctl_clean);
void launch_tc_assemble(scw_ctx* ctx, const scw_layer* L, int64_t Fz, const double* z, void* P, int64_t ldP,
                        void* scratch);
// Generic complex64 GEMM on the assembly kernel (BF16x3 tcgen05): C [ldC x N] col-major = A [ldA x K] col-major (R rows,
// 16-byte aligned) . B [K x N] row-major; scratch = tc_assemble_scratch(ctx, R, K, N, 1).
void launch_tc_gemm(scw_ctx* ctx, int64_t R, int64_t K, int64_t N, const void* A, int64_t ldA, const void* B, void* C,
                    int64_t ldC, void* scratch);

// ---- scw_vbuild.cu: V = T Q diag(alpha), eq. 33 (NEXT-2) -------------------------------------------------------
size_t vbuild_scratch(const scw_ctx* ctx, const scw_vbuild* vb);
void launch_vbuild(scw_ctx* ctx, const scw_vbuild* vb, void* V, int64_t ldV, void* scratch);

// Detector reductions of a sweep (NEXT-3): what leaves the synthesis instead of the complex field.
struct TcDetector {
    void* const* I;        // per instance: real [Fz][Ny][Nx] at s3 strides (passed as strides[1..3]), or NULL: not wanted
    void* const* S;        // per instance: real [Fz] sums of I over the window, or NULL: not wanted
    int64_t win[4];        // ix0, ix1, iy0, iy1 (grid indices, half-open)
    void* s_part;          // scratch of tc_synth_wsum_bytes() for the fused kernel (when S is wanted)
};

// ---- scw_tc_synth.cu: tcgen05 BF16x3 separable synthesis (complex64, 2U and 2V <= 80) ---------------
bool tc_synth_supported(int dtype, int U, int Vn);
size_t tc_synth_twiddle_bytes(int U, int Vn, int64_t Nx, int64_t Ny);
size_t tc_synth_scratch(int U, int Vn, int64_t Fz);
// zero/n_zero: ints cleared by the same launch (the control block of the assembly that follows), may be NULL
void launch_tc_synth_twiddles(scw_ctx* ctx, int U, int Vn, double X, double Y, int64_t Nx, const double* x, int64_t Ny,
                              const double* y, void* tw, int* zero = nullptr, size_t n_zero = 0);
int tc_synth_max_group();
// Image layout of a synthesis over `scratch` (for the assembly's fix-up) and its plane counters inside the twiddle blob.
void tc_synth_image_plan(int U, int Vn, int64_t Nx, int64_t Ny, void* scratch, const void* tw, TcFixup* fix, int** sched,
                         int* n_sched);
// n_inst instances with equal Fz, spectra back to back in P_all ([ldP x n_inst*Fz]); scratch = tc_synth_scratch(U, Vn, Fz*n_inst)
// det != NULL: detector mode (no complex field; I at z*strides[1] + y*strides[2] + x*strides[3] and / or window sums)
void launch_tc_synth_group(scw_ctx* ctx, int U, int Vn, int64_t Fz, int n_inst, const void* P_all, int64_t ldP,
                           int64_t Nx, int64_t Ny, const void* tw, void* const* E, const int64_t strides[4],
                           void* scratch, const TcDetector* det = nullptr);
size_t tc_synth_wsum_bytes(int64_t planes_z, int64_t Nx, int64_t Ny);
// Same, with the spectrum images already in `scratch` and the plane counters zeroed (written by the assembly's fix-up).
void launch_tc_synth_group_images(scw_ctx* ctx, int U, int Vn, int64_t Fz, int n_inst, int64_t Nx, int64_t Ny,
                                  const void* tw, void* const* E, const int64_t strides[4], void* scratch,
                                  const TcDetector* det = nullptr);
void launch_tc_synth(scw_ctx* ctx, int U, int Vn, int64_t Fz, const void* P, int64_t ldP, int64_t Nx, int64_t Ny,
                     const void* tw, void* E, const int64_t strides[4], void* scratch);
// Exterior field (eq. 9-10) on a grid, complex64: spectrum images from eq. 9 directly, then the synthesis; scratch = tc_synth_scratch(U, Vn, Fz)
void launch_tc_synth_exterior(scw_ctx* ctx, const scw_exterior* e, int64_t Fz, const double* z, int64_t Nx, int64_t Ny,
                              const void* tw, void* E, const int64_t strides[4], void* scratch);

// ---- scw_dmma.cu: FP64 tensor-core (DMMA mma.sync) batched complex GEMM for the complex128 contractions -----------
bool dmma_supported(int dtype);
size_t dmma_assemble_scratch(int64_t R, int64_t J, int64_t Fz, int sm_count);
// P = V W with W[j*Fz + i] from launch_mode_weights; scratch from dmma_assemble_scratch
void launch_dmma_assemble(scw_ctx* ctx, int64_t R, int64_t J, int64_t Fz, const void* V, int64_t ldV, const void* W,
                          void* P, int64_t ldP, void* scratch);
// two-pass synthesis with the frequency-major tables of launch_twiddles; scratch = simt_synth_scratch(SCW_C128, ...)
void launch_dmma_synth(scw_ctx* ctx, int U, int Vn, int64_t Fz, const void* P, int64_t ldP, int64_t Nx, const void* FxT,
                       int64_t Ny, const void* FyT, void* E, const int64_t strides[4], void* scratch);

void launch_dmma_gemm_sub(scw_ctx* ctx, int64_t M, int64_t N, int64_t K, const void* A, int64_t ldA, const void* B, int64_t ldB,
                          void* C, int64_t ldC);

// ---- scw_alpha.cu: alpha propagation across layers, eq. 24-26 (NEXT-4) -------------------------------------------
bool alpha_supported(const scw_ctx* ctx, int64_t n);
size_t alpha_scratch(const scw_ctx* ctx, int64_t n);
void launch_propagate_alpha(scw_ctx* ctx, const scw_stack* st, const void* r0, void* const* alpha, void* rL, void* scratch);

// ---- scw_exterior.cu: eq. 9 in the half-spaces above / below the sample (NEXT-1) -------------------------------
void launch_exterior_spectra(scw_ctx* ctx, const scw_exterior* e, int64_t Fz, const double* z, void* P, int64_t ldP);
size_t exterior_points_bytes(const scw_exterior* e);
void launch_exterior_points(scw_ctx* ctx, const scw_exterior* e, int64_t N, const double* r, void* E, void* ws);

// ---- points.cu ------------------------------------------------------------------------------
struct PwTableInfo { size_t bytes; };
size_t points_table_bytes(int dtype, int64_t J);
void launch_points_planewave(scw_ctx* ctx, const scw_modes* m, int64_t N, const double* r, void* E,
                             void* table);
// same sum with the table in the library's built-in array (scw_eval_points_noalloc): allocates nothing; returns the CUDA
// error of the address look-up / memset, launch errors are left for cudaGetLastError
cudaError_t launch_points_planewave_noalloc(scw_ctx* ctx, const scw_modes* m, int64_t N, const double* r, void* E);
// dense form, per-point synthesis: E[p,comp] = sum_m P[comp*M+m, p] exp(i 2 pi (u x_p/X + v y_p/Y))
void launch_point_synth(scw_ctx* ctx, int dtype, int U, int Vn, double X, double Y, int64_t n,
                        const double* r, const void* P, int64_t ldP, void* E);
// z[p] = r[3p+2]
void launch_extract_z(scw_ctx* ctx, int64_t n, const double* r, double* z);

}  // namespace scw
