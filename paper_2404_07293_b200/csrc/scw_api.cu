// C ABI of libscw: argument validation, workspace carving and kernel dispatch.
// See include/scwatter.h for the contract of every entry point.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "scw_internal.h"

using namespace scw;

namespace {

int32_t fail(scw_ctx* ctx, int32_t code, const char* fmt, ...)
{
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->msg, sizeof(ctx->msg), fmt, ap);
        va_end(ap);
    }
    return code;
}

inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }
inline size_t esize(int dtype) { return dtype == SCW_C64 ? 8 : 16; }
inline bool finite_pos(double v) { return std::isfinite(v) && v > 0.0; }

constexpr int64_t MAX_FREQ = 4096;        // per-axis frequency count
constexpr int64_t MAX_GRID = 1 << 20;     // per-axis grid points

// sweep_call: only back-to-back sweep calls keep the cached twiddles / clean control block (any other call may carve
// the same workspace bytes differently)
int32_t check_ctx(scw_ctx* ctx, bool sweep_call = false)
{
    if (!ctx) return SCW_ERR_NULL;
    if (!sweep_call) {
        ctx->tw_valid = false;
        ctx->clean_ctl = nullptr;
        ctx->clean_img = nullptr;
    }
    ctx->msg[0] = 0;
    ctx->cuda_err = 0;
    ctx->required_ws = 0;
    ctx->tc_error = false;
    ctx->last_classes = 0;
    ctx->prof_last = nullptr;       // per-kernel timers: the first kernel of this call gets its own start event
    ctx->tl_ring = nullptr;         // timeline ring: set by the assembly launch of this call, if any
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e == cudaSuccess && cur != ctx->device) e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) {
        ctx->cuda_err = (int32_t)e;
        return fail(ctx, SCW_ERR_CUDA, "cudaSetDevice(%d): %s", ctx->device, cudaGetErrorString(e));
    }
    return SCW_OK;
}

int32_t check_launch(scw_ctx* ctx, const char* what)
{
    if (ctx->tc_error) return fail(ctx, SCW_ERR_CUDA, "%s: cuTensorMapEncodeTiled failed", what);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        ctx->cuda_err = (int32_t)e;
        return fail(ctx, SCW_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
    }
    return SCW_OK;
}

int32_t check_layer(scw_ctx* ctx, const scw_layer* L, const char* who)
{
    if (!L) return fail(ctx, SCW_ERR_NULL, "%s: layer is NULL", who);
    if (L->struct_size != sizeof(scw_layer))
        return fail(ctx, SCW_ERR_SHAPE, "%s: layer.struct_size %u != %zu", who, L->struct_size, sizeof(scw_layer));
    if (L->dtype != SCW_C64 && L->dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "%s: bad dtype %d", who, L->dtype);
    if (L->U <= 0 || L->Vn <= 0 || L->U > MAX_FREQ || L->Vn > MAX_FREQ)
        return fail(ctx, SCW_ERR_SHAPE, "%s: U=%d Vn=%d out of range", who, L->U, L->Vn);
    if (L->J <= 0) return fail(ctx, SCW_ERR_SHAPE, "%s: J=%lld must be positive", who, (long long)L->J);
    const int64_t R = 3LL * L->U * L->Vn;
    if (L->ldV < R) return fail(ctx, SCW_ERR_SHAPE, "%s: ldV=%lld < 3*U*Vn=%lld", who, (long long)L->ldV, (long long)R);
    if (!finite_pos(L->X) || !finite_pos(L->Y) || !finite_pos(L->lambda))
        return fail(ctx, SCW_ERR_VALUE, "%s: X, Y and lambda must be finite and > 0", who);
    if (!std::isfinite(L->z_lo) || !std::isfinite(L->z_hi) || L->z_hi < L->z_lo)
        return fail(ctx, SCW_ERR_VALUE, "%s: need finite z_lo <= z_hi", who);
    if (!L->V || !L->gamma) return fail(ctx, SCW_ERR_NULL, "%s: V and gamma are required", who);
    const size_t es = esize(L->dtype);
    if (!aligned(L->V, es) || (L->c && !aligned(L->c, es)) || !aligned(L->gamma, 16))
        return fail(ctx, SCW_ERR_ALIGN, "%s: V/c/gamma misaligned", who);
    return SCW_OK;
}

int32_t need_ws(scw_ctx* ctx, size_t bytes, const char* who)
{
    if (bytes == 0) return SCW_OK;
    if (!ctx->ws || ctx->ws_bytes < bytes) {
        ctx->required_ws = bytes;
        return fail(ctx, SCW_ERR_WORKSPACE, "%s: workspace of %zu bytes required, %zu registered", who, bytes,
                    ctx->ws_bytes);
    }
    return SCW_OK;
}

// ---- assembly -----------------------------------------------------------------------------
// Tensor-core assembly is used for complex64 unless the ctx is pinned to the CUDA-core path; tiny
// problems (less than one 128 x 64 tile) stay on CUDA cores in AUTO mode.
bool use_tc_assemble(const scw_ctx* ctx, const scw_layer* L, int64_t Fz)
{
    const int64_t R = 3LL * L->U * L->Vn;
    if (ctx->path == SCW_PATH_SIMT || !tc_assemble_supported(L->dtype, R, L->J, Fz, L->V, L->ldV)) return false;
    if (ctx->path == SCW_PATH_TENSOR) return true;
    return 2 * R >= 128 && L->J >= 64;
}

// complex128 runs on the FP64 tensor cores (DMMA) unless the ctx is pinned to the CUDA-core path
bool use_dmma(const scw_ctx* ctx, int dtype) { return ctx->path != SCW_PATH_SIMT && dmma_supported(dtype); }

size_t assemble_ws(const scw_ctx* ctx, const scw_layer* L, int64_t Fz)
{
    const int64_t R = 3LL * L->U * L->Vn;
    if (use_tc_assemble(ctx, L, Fz)) return tc_assemble_scratch(ctx, R, L->J, Fz, 1);
    if (use_dmma(ctx, L->dtype))
        return align_up((size_t)L->J * Fz * esize(L->dtype)) + dmma_assemble_scratch(R, L->J, Fz, ctx->sm_count);
    return align_up((size_t)L->J * Fz * esize(L->dtype)) + simt_assemble_scratch(L->dtype, R, L->J, Fz, ctx->sm_count);
}

void run_assemble(scw_ctx* ctx, const scw_layer* L, int64_t Fz, const double* z, void* P, int64_t ldP, Carver& cv)
{
    const int64_t R = 3LL * L->U * L->Vn;
    if (use_tc_assemble(ctx, L, Fz)) {
        void* scratch = cv.take(tc_assemble_scratch(ctx, R, L->J, Fz, 1));
        launch_tc_assemble(ctx, L, Fz, z, P, ldP, scratch);
        return;
    }
    // the weights and the scratch of these paths go where a tensor-core assembly over the same carver keeps its control
    // block (per-instance sweeps alternate between them): that block is no longer known clean
    ctx->clean_ctl = nullptr;
    void* W = cv.take((size_t)L->J * Fz * esize(L->dtype));
    if (use_dmma(ctx, L->dtype)) {
        void* scratch = cv.take(dmma_assemble_scratch(R, L->J, Fz, ctx->sm_count));
        launch_mode_weights(ctx, L->dtype, L->J, Fz, L->lambda, L->z_lo, L->z_hi, L->c, L->gamma, L->dir, z, W);
        launch_dmma_assemble(ctx, R, L->J, Fz, L->V, L->ldV, W, P, ldP, scratch);
        return;
    }
    void* scratch = cv.take(simt_assemble_scratch(L->dtype, R, L->J, Fz, ctx->sm_count));
    launch_mode_weights(ctx, L->dtype, L->J, Fz, L->lambda, L->z_lo, L->z_hi, L->c, L->gamma, L->dir, z, W);
    launch_simt_assemble(ctx, L->dtype, R, L->J, Fz, L->V, L->ldV, W, P, ldP, scratch);
}

// ---- synthesis ----------------------------------------------------------------------------
// ---- synthesis: tensor-core kernel for complex64 with 2U, 2V <= 80, CUDA-core kernels otherwise ----
bool use_tc_synth(const scw_ctx* ctx, int dtype, int U, int Vn)
{
    return ctx->path != SCW_PATH_SIMT && tc_synth_supported(dtype, U, Vn);
}

struct Twiddles {
    bool tc;
    void* a;     // CUDA-core: FxT [U x Nx];  tensor-core: image blob (A1 | A2)
    void* b;     // CUDA-core: FyT [Vn x Ny]
};

size_t twiddle_ws(const scw_ctx* ctx, int dtype, int U, int Vn, int64_t Nx, int64_t Ny)
{
    if (use_tc_synth(ctx, dtype, U, Vn)) return align_up(tc_synth_twiddle_bytes(U, Vn, Nx, Ny));
    return align_up((size_t)U * Nx * esize(dtype)) + align_up((size_t)Vn * Ny * esize(dtype));
}

size_t synth_ws(const scw_ctx* ctx, int dtype, int U, int Vn, int64_t Fz, int64_t Ny)
{
    if (use_tc_synth(ctx, dtype, U, Vn)) return align_up(tc_synth_scratch(U, Vn, Fz));
    return simt_synth_scratch(dtype, U, Fz, Ny);
}

// a-3.  With SCW_OPT_CACHE on, the tables of the previous call are reused when the key (coordinate pointers, sizes,
// frequency grid, periods, location in the workspace) is unchanged.  zero / n_zero: ints the tensor-core twiddle kernel
// clears on the way (control block of the assembly that follows); *zeroed tells whether that happened.
Twiddles run_twiddles(scw_ctx* ctx, int dtype, int U, int Vn, double X, double Y, int64_t Nx, const double* x,
                      int64_t Ny, const double* y, Carver& cv, int* zero = nullptr, size_t n_zero = 0, bool* zeroed = nullptr)
{
    Twiddles t;
    t.tc = use_tc_synth(ctx, dtype, U, Vn);
    if (zeroed) *zeroed = false;
    if (t.tc) {
        t.a = cv.take(tc_synth_twiddle_bytes(U, Vn, Nx, Ny));
        t.b = nullptr;
    } else {
        t.a = cv.take((size_t)U * Nx * esize(dtype));
        t.b = cv.take((size_t)Vn * Ny * esize(dtype));
    }
    scw_ctx::TwKey key;
    key.x = x; key.y = y; key.where = t.a; key.Nx = Nx; key.Ny = Ny; key.U = U; key.Vn = Vn; key.dtype = dtype;
    key.X = X; key.Y = Y; key.tc = t.tc;
    const scw_ctx::TwKey& k0 = ctx->tw_key;
    if (ctx->cache_on && ctx->tw_valid && k0.x == key.x && k0.y == key.y && k0.where == key.where && k0.Nx == key.Nx &&
        k0.Ny == key.Ny && k0.U == key.U && k0.Vn == key.Vn && k0.dtype == key.dtype && k0.X == key.X && k0.Y == key.Y &&
        k0.tc == key.tc)
        return t;
    if (t.tc) {
        launch_tc_synth_twiddles(ctx, U, Vn, X, Y, Nx, x, Ny, y, t.a, zero, n_zero);
        if (zeroed) *zeroed = zero != nullptr;
    } else {
        launch_twiddles(ctx, dtype, U, Nx, x, X, t.a);
        launch_twiddles(ctx, dtype, Vn, Ny, y, Y, t.b);
    }
    ctx->tw_key = key;
    ctx->tw_valid = ctx->cache_on;
    return t;
}

void run_synth(scw_ctx* ctx, const Twiddles& t, int dtype, int U, int Vn, int64_t Fz, const void* P, int64_t ldP,
               int64_t Nx, int64_t Ny, void* E, const int64_t s4[4], void* scratch)
{
    if (t.tc) launch_tc_synth(ctx, U, Vn, Fz, P, ldP, Nx, Ny, t.a, E, s4, scratch);
    else if (use_dmma(ctx, dtype)) launch_dmma_synth(ctx, U, Vn, Fz, P, ldP, Nx, t.a, Ny, t.b, E, s4, scratch);
    else launch_simt_synth(ctx, dtype, U, Vn, Fz, P, ldP, Nx, t.a, Ny, t.b, E, s4, scratch);
}

int32_t check_grid(scw_ctx* ctx, int32_t dtype, int32_t U, int32_t Vn, double X, double Y, int64_t Nx,
                   const double* x, int64_t Ny, const double* y, const char* who)
{
    if (dtype != SCW_C64 && dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "%s: bad dtype %d", who, dtype);
    if (U <= 0 || Vn <= 0 || U > MAX_FREQ || Vn > MAX_FREQ) return fail(ctx, SCW_ERR_SHAPE, "%s: U=%d Vn=%d out of range", who, U, Vn);
    if (Nx <= 0 || Ny <= 0 || Nx > MAX_GRID || Ny > MAX_GRID)
        return fail(ctx, SCW_ERR_SHAPE, "%s: Nx=%lld Ny=%lld out of range", who, (long long)Nx, (long long)Ny);
    if (!finite_pos(X) || !finite_pos(Y)) return fail(ctx, SCW_ERR_VALUE, "%s: X and Y must be finite and > 0", who);
    if (!x || !y) return fail(ctx, SCW_ERR_NULL, "%s: x and y are required", who);
    if (!aligned(x, 8) || !aligned(y, 8)) return fail(ctx, SCW_ERR_ALIGN, "%s: x/y misaligned", who);
    return SCW_OK;
}

void planar_strides(int64_t Nx, int64_t Ny, int64_t s[4])
{
    s[3] = 1;
    s[2] = Nx;
    s[0] = Nx * Ny;
    s[1] = 3 * Nx * Ny;
}

}  // namespace

extern "C" {

int32_t scw_version(void) { return 100; }

int32_t scw_create(scw_ctx** out, int32_t device, void* cuda_stream)
{
    if (!out) return SCW_ERR_NULL;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return SCW_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return SCW_ERR_CUDA;
    if (prop.major != 10) return SCW_ERR_UNSUPPORTED;
    scw_ctx* ctx = new (std::nothrow) scw_ctx();
    if (!ctx) return SCW_ERR_CUDA;
    ctx->device = device;
    ctx->sm_count = prop.multiProcessorCount;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    *out = ctx;
    return SCW_OK;
}

int32_t scw_destroy(scw_ctx* ctx)
{
    if (!ctx) return SCW_ERR_NULL;
    for (ProfRec& r : ctx->recs) { if (r.owns_a) cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    if (ctx->h2d_stream) cudaStreamDestroy(ctx->h2d_stream);
    if (ctx->d2h_stream) cudaStreamDestroy(ctx->d2h_stream);
    if (ctx->ev_start) cudaEventDestroy(ctx->ev_start);
    for (int b = 0; b < 2; ++b) {
        if (ctx->ev_in[b]) cudaEventDestroy(ctx->ev_in[b]);
        if (ctx->ev_done[b]) cudaEventDestroy(ctx->ev_done[b]);
        if (ctx->ev_out[b]) cudaEventDestroy(ctx->ev_out[b]);
    }
    delete ctx;
    return SCW_OK;
}

int32_t scw_set_stream(scw_ctx* ctx, void* cuda_stream)
{
    if (!ctx) return SCW_ERR_NULL;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    return SCW_OK;
}

int32_t scw_set_workspace(scw_ctx* ctx, void* dev_ptr, size_t bytes)
{
    if (!ctx) return SCW_ERR_NULL;
    if ((dev_ptr == nullptr) != (bytes == 0)) return fail(ctx, SCW_ERR_NULL, "workspace pointer/size mismatch");
    if (!aligned(dev_ptr, 256)) return fail(ctx, SCW_ERR_ALIGN, "workspace must be 256-byte aligned");
    ctx->ws = dev_ptr;
    ctx->ws_bytes = bytes;
    ctx->tw_valid = false;
    ctx->clean_ctl = nullptr;
    ctx->clean_img = nullptr;
    // the per-CTA timers and the timeline ring of the last assembly lived in the previous workspace, which the caller may
    // free now: scw_profile_assembly / scw_profile_timeline report "nothing recorded" until the next launch
    ctx->last_asm_ns = nullptr;
    ctx->last_asm_G = 0;
    ctx->tl_last_ring = nullptr;
    ctx->tl_ring = nullptr;
    ctx->tl_seq = 0;
    return SCW_OK;
}

int32_t scw_invalidate_cache(scw_ctx* ctx)
{
    if (!ctx) return SCW_ERR_NULL;
    ctx->tw_valid = false;
    ctx->clean_ctl = nullptr;
    ctx->clean_img = nullptr;
    return SCW_OK;
}

int32_t scw_set_option(scw_ctx* ctx, int32_t option, int64_t value)
{
    if (!ctx) return SCW_ERR_NULL;
    if (option == SCW_OPT_PATH && value >= SCW_PATH_AUTO && value <= SCW_PATH_TENSOR) {
        ctx->path = value;
        ctx->tw_valid = false;
        ctx->clean_ctl = nullptr;       // the other path carves the same workspace bytes differently
        ctx->clean_img = nullptr;
        return SCW_OK;
    }
    if (option == SCW_OPT_CACHE && (value == 0 || value == 1)) {
        ctx->cache_on = value != 0;
        ctx->tw_valid = false;
        ctx->clean_ctl = nullptr;
        ctx->clean_img = nullptr;
        return SCW_OK;
    }
    if (option == SCW_OPT_PROFILE && (value == 0 || value == 1)) {
        ctx->profile = value != 0;
        return SCW_OK;
    }
    return fail(ctx, SCW_ERR_UNSUPPORTED, "unknown option %d / value %lld", option, (long long)value);
}

int32_t scw_profile_classes(void) { return KC_COUNT; }

const char* scw_profile_name(int32_t kc)
{
    static const char* names[KC_COUNT] = {"mode_weights", "twiddles", "simt_assemble", "reduce_splits", "simt_synth_a",
                                          "simt_synth_b", "points_table", "points_planewave", "point_synth", "misc",
                                          "tc_assemble", "tc_synth", "tc_synth_images", "dmma_assemble", "dmma_synth_a",
                                          "dmma_synth_b", "exterior", "vbuild_prepare", "alpha_misc", "alpha_lu_update", "alpha_lu_panel"};
    return (kc >= 0 && kc < KC_COUNT) ? names[kc] : nullptr;
}

static void profile_drain(scw_ctx* ctx)
{
    for (ProfRec& r : ctx->recs) {
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) == cudaSuccess && cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) {
            ctx->prof_ms[r.kc] += (double)ms;
            ctx->prof_n[r.kc] += 1;
        }
    }
    for (ProfRec& r : ctx->recs) {                     // a record's start event may be its predecessor's end event
        if (r.owns_a) cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    ctx->recs.clear();
    ctx->prof_last = nullptr;
}

int32_t scw_profile_read(scw_ctx* ctx, int32_t kc, double* ms_total, int64_t* launches)
{
    if (!ctx) return SCW_ERR_NULL;
    if (kc < 0 || kc >= KC_COUNT) return fail(ctx, SCW_ERR_SHAPE, "kernel class %d out of range", kc);
    profile_drain(ctx);
    if (ms_total) *ms_total = ctx->prof_ms[kc];
    if (launches) *launches = ctx->prof_n[kc];
    return SCW_OK;
}

int32_t scw_profile_reset(scw_ctx* ctx)
{
    if (!ctx) return SCW_ERR_NULL;
    profile_drain(ctx);
    for (int i = 0; i < KC_COUNT; ++i) { ctx->prof_ms[i] = 0; ctx->prof_n[i] = 0; }
    return SCW_OK;
}

const char* scw_last_error(const scw_ctx* ctx) { return ctx ? ctx->msg : "ctx is NULL"; }
int32_t scw_last_cuda_error(const scw_ctx* ctx) { return ctx ? ctx->cuda_err : 0; }
size_t scw_required_workspace(const scw_ctx* ctx) { return ctx ? ctx->required_ws : 0; }
int64_t scw_launch_count(const scw_ctx* ctx) { return ctx ? ctx->launches : 0; }
uint64_t scw_last_kernels(const scw_ctx* ctx) { return ctx ? ctx->last_classes : 0; }

// ------------------------------------------------------------------------------------------
int32_t scw_assemble_workspace(scw_ctx* ctx, const scw_layer* layer, int64_t Fz, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    if (int32_t s = check_layer(ctx, layer, "scw_assemble_workspace")) return s;
    if (Fz < 0) return fail(ctx, SCW_ERR_SHAPE, "Fz=%lld < 0", (long long)Fz);
    *bytes = Fz ? assemble_ws(ctx, layer, Fz) : 0;
    return SCW_OK;
}

int32_t scw_assemble_spectra(scw_ctx* ctx, const scw_layer* layer, int64_t Fz, const double* z, void* P, int64_t ldP)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_layer(ctx, layer, "scw_assemble_spectra")) return s;
    if (Fz < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_assemble_spectra: Fz=%lld < 0", (long long)Fz);
    if (Fz == 0) return SCW_OK;
    if (!z || !P) return fail(ctx, SCW_ERR_NULL, "scw_assemble_spectra: z and P are required");
    const int64_t R = 3LL * layer->U * layer->Vn;
    if (ldP < R) return fail(ctx, SCW_ERR_SHAPE, "scw_assemble_spectra: ldP=%lld < 3*U*Vn=%lld", (long long)ldP, (long long)R);
    if (!aligned(z, 8) || !aligned(P, esize(layer->dtype))) return fail(ctx, SCW_ERR_ALIGN, "scw_assemble_spectra: z/P misaligned");
    if (int32_t s = need_ws(ctx, assemble_ws(ctx, layer, Fz), "scw_assemble_spectra")) return s;
    Carver cv(ctx->ws);
    run_assemble(ctx, layer, Fz, z, P, ldP, cv);
    return check_launch(ctx, "scw_assemble_spectra");
}

// ------------------------------------------------------------------------------------------
int32_t scw_synthesize_workspace(scw_ctx* ctx, int32_t dtype, int32_t U, int32_t Vn, int64_t Fz, int64_t Nx,
                                 int64_t Ny, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    if (dtype != SCW_C64 && dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "bad dtype %d", dtype);
    if (U <= 0 || Vn <= 0 || Fz < 0 || Nx <= 0 || Ny <= 0) return fail(ctx, SCW_ERR_SHAPE, "bad dimensions");
    *bytes = Fz ? twiddle_ws(ctx, dtype, U, Vn, Nx, Ny) + synth_ws(ctx, dtype, U, Vn, Fz, Ny) : 0;
    return SCW_OK;
}

int32_t scw_synthesize_grid(scw_ctx* ctx, int32_t dtype, int32_t U, int32_t Vn, double X, double Y, int64_t Fz,
                            const void* P, int64_t ldP, int64_t Nx, const double* x, int64_t Ny, const double* y,
                            void* E, const int64_t* strides)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_grid(ctx, dtype, U, Vn, X, Y, Nx, x, Ny, y, "scw_synthesize_grid")) return s;
    if (Fz < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_synthesize_grid: Fz=%lld < 0", (long long)Fz);
    if (Fz == 0) return SCW_OK;
    if (!P || !E) return fail(ctx, SCW_ERR_NULL, "scw_synthesize_grid: P and E are required");
    if (ldP < 3LL * U * Vn) return fail(ctx, SCW_ERR_SHAPE, "scw_synthesize_grid: ldP=%lld < 3*U*Vn", (long long)ldP);
    if (!aligned(P, esize(dtype)) || !aligned(E, esize(dtype))) return fail(ctx, SCW_ERR_ALIGN, "scw_synthesize_grid: P/E misaligned");
    int64_t s4[4];
    if (strides) memcpy(s4, strides, sizeof(s4)); else planar_strides(Nx, Ny, s4);
    for (int i = 0; i < 4; ++i)
        if (s4[i] < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_synthesize_grid: negative stride");
    if (ctx->path == SCW_PATH_TENSOR && !tc_synth_supported(dtype, U, Vn) && !dmma_supported(dtype))
        return fail(ctx, SCW_ERR_UNSUPPORTED, "scw_synthesize_grid: no tensor-core synthesis for this dtype / frequency count");
    if (int32_t s = need_ws(ctx, twiddle_ws(ctx, dtype, U, Vn, Nx, Ny) + synth_ws(ctx, dtype, U, Vn, Fz, Ny), "scw_synthesize_grid")) return s;
    Carver cv(ctx->ws);
    const Twiddles tw = run_twiddles(ctx, dtype, U, Vn, X, Y, Nx, x, Ny, y, cv);
    void* scratch = cv.take(synth_ws(ctx, dtype, U, Vn, Fz, Ny));
    run_synth(ctx, tw, dtype, U, Vn, Fz, P, ldP, Nx, Ny, E, s4, scratch);
    return check_launch(ctx, "scw_synthesize_grid");
}

// ------------------------------------------------------------------------------------------
static int32_t check_sweep(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t Nx,
                           int64_t Ny, const char* who, int64_t* fz_max, size_t* asm_max)
{
    if (n_inst < 0) return fail(ctx, SCW_ERR_SHAPE, "%s: n_inst=%lld < 0", who, (long long)n_inst);
    if (n_inst == 0) return SCW_OK;
    if (!inst || !Fz) return fail(ctx, SCW_ERR_NULL, "%s: inst and Fz are required", who);
    if (Nx <= 0 || Ny <= 0 || Nx > MAX_GRID || Ny > MAX_GRID) return fail(ctx, SCW_ERR_SHAPE, "%s: bad Nx/Ny", who);
    *fz_max = 0;
    *asm_max = 0;
    for (int64_t i = 0; i < n_inst; ++i) {
        if (int32_t s = check_layer(ctx, &inst[i], who)) return s;
        if (inst[i].dtype != inst[0].dtype || inst[i].U != inst[0].U || inst[i].Vn != inst[0].Vn ||
            inst[i].X != inst[0].X || inst[i].Y != inst[0].Y)
            return fail(ctx, SCW_ERR_SHAPE, "%s: instance %lld differs in dtype/U/Vn/X/Y", who, (long long)i);
        if (Fz[i] < 0) return fail(ctx, SCW_ERR_SHAPE, "%s: Fz[%lld] < 0", who, (long long)i);
        if (Fz[i] > *fz_max) *fz_max = Fz[i];
        if (Fz[i] > 0) {
            // the scratch size is a function of (J, Fz, path eligibility) once U, Vn, dtype are equal: instances of a sweep
            // mostly repeat the previous one's shape, and planning the stream-K split 64 times per call showed on the host
            const bool tc = use_tc_assemble(ctx, &inst[i], Fz[i]);
            if (i == 0 || inst[i].J != inst[i - 1].J || Fz[i] != Fz[i - 1] || Fz[i - 1] <= 0 ||
                tc != use_tc_assemble(ctx, &inst[i - 1], Fz[i - 1])) {
                const size_t a = assemble_ws(ctx, &inst[i], Fz[i]);
                if (a > *asm_max) *asm_max = a;
            }
        }
    }
    return SCW_OK;
}

// Grouped (batched) sweep: every instance on the tensor-core kernels with the same J and Fz.
// Grouped (batched) sweep: every instance on the tensor-core kernels.  The instances are cut into runs of consecutive
// instances with the same J and Fz (at most 64 per run): each run is ONE assembly launch and ONE synthesis launch.
// Empty = the sweep takes the per-instance path (some instance cannot run on the tensor-core kernels, or has Fz = 0).
struct SweepRun { int64_t i0; int n; };

static std::vector<SweepRun> sweep_runs(const scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz)
{
    std::vector<SweepRun> runs;
    if (n_inst < 1 || !use_tc_synth(ctx, inst[0].dtype, inst[0].U, inst[0].Vn)) return runs;
    const int gmax = tc_assemble_max_group() < tc_synth_max_group() ? tc_assemble_max_group() : tc_synth_max_group();
    for (int64_t i = 0; i < n_inst; ++i) {          // every instance must be able to take the TMA path (16-byte aligned V, ...)
        if (Fz[i] <= 0 || !use_tc_assemble(ctx, &inst[i], Fz[i])) return std::vector<SweepRun>();
        if (!runs.empty() && runs.back().n < gmax && inst[i].J == inst[runs.back().i0].J && Fz[i] == Fz[runs.back().i0])
            runs.back().n++;
        else
            runs.push_back(SweepRun{i, 1});
    }
    return runs;
}

static size_t sweep_ws(const scw_ctx* ctx, const scw_layer* L0, int64_t fz_max, size_t asm_max, int64_t Nx, int64_t Ny)
{
    if (fz_max == 0) return 0;
    const int64_t R = 3LL * L0->U * L0->Vn;
    return twiddle_ws(ctx, L0->dtype, L0->U, L0->Vn, Nx, Ny) + align_up((size_t)R * fz_max * esize(L0->dtype)) + asm_max +
           synth_ws(ctx, L0->dtype, L0->U, L0->Vn, fz_max, Ny);
}

// workspace of a sweep; the general (non-grouped) detector path adds a planar E buffer for one instance
// Detector reductions asked of a sweep (NEXT-3): per-sample intensity I and / or its sum S over a window of every plane.
struct DetArgs {
    void* const* I;
    void* const* S;
    int64_t win[4];     // ix0, ix1, iy0, iy1
};

static size_t sweep_need(const scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t fz_max,
                         size_t asm_max, int64_t Nx, int64_t Ny, const DetArgs* det)
{
    if (!n_inst || fz_max == 0) return 0;
    const std::vector<SweepRun> runs = sweep_runs(ctx, n_inst, inst, Fz);
    if (!runs.empty()) {                            // twiddles | assembly scratch | images | window partials, each sized for the largest run
        size_t a = 0, sy = 0, w = 0;
        const int64_t R = 3LL * inst[0].U * inst[0].Vn;
        for (const SweepRun& r : runs) {
            a = std::max(a, align_up(tc_assemble_scratch(ctx, R, inst[r.i0].J, Fz[r.i0], r.n)));
            sy = std::max(sy, align_up(tc_synth_scratch(inst[0].U, inst[0].Vn, Fz[r.i0] * r.n)));
            if (det) w = std::max(w, tc_synth_wsum_bytes(Fz[r.i0] * r.n, Nx, Ny));
        }
        return twiddle_ws(ctx, inst[0].dtype, inst[0].U, inst[0].Vn, Nx, Ny) + a + sy + w;
    }
    return sweep_ws(ctx, &inst[0], fz_max, asm_max, Nx, Ny) +
           (det ? align_up((size_t)fz_max * 3 * Nx * Ny * esize(inst[0].dtype)) : 0);
}

static int32_t sweep_workspace_impl(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t Nx,
                                    int64_t Ny, size_t* bytes, bool detector, const char* who)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    int64_t fz_max = 0;
    size_t asm_max = 0;
    if (int32_t s = check_sweep(ctx, n_inst, inst, Fz, Nx, Ny, who, &fz_max, &asm_max)) return s;
    const DetArgs any = {};
    *bytes = sweep_need(ctx, n_inst, inst, Fz, fz_max, asm_max, Nx, Ny, detector ? &any : nullptr);
    return SCW_OK;
}

int32_t scw_sweep_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t Nx,
                            int64_t Ny, size_t* bytes)
{
    return sweep_workspace_impl(ctx, n_inst, inst, Fz, Nx, Ny, bytes, false, "scw_sweep_workspace");
}

int32_t scw_sweep_intensity_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t Nx,
                                      int64_t Ny, size_t* bytes)
{
    return sweep_workspace_impl(ctx, n_inst, inst, Fz, Nx, Ny, bytes, true, "scw_sweep_intensity_workspace");
}

// Shared by the device- and host-buffer variants: everything after validation.
static void run_sweep(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, const double* const* z,
                      int64_t Nx, const double* x, int64_t Ny, const double* y, void* const* E, const int64_t s4[4],
                      int64_t fz_max, size_t asm_max, Carver& cv, const DetArgs* det = nullptr)
{
    // det: no complex field; det->I[i] are real buffers receiving sum_comp |E_comp|^2 at n*s4[1] + k*s4[2] + i*s4[3], det->S[i]
    // the window sums (NEXT-3)
    const scw_layer& L0 = inst[0];
    const int64_t R = 3LL * L0.U * L0.Vn;
    const std::vector<SweepRun> runs = sweep_runs(ctx, n_inst, inst, Fz);
    if (!runs.empty()) {
        // batched: all instances of a run go through ONE assembly launch (weights + P = V W + fix-up that writes the
        // synthesis kernel's spectrum images: P never goes to memory) and ONE synthesis launch; the twiddle launch, when
        // it is not served from the cache, also clears the assembly's control block
        size_t a_max = 0, s_max = 0, w_max = 0;
        for (const SweepRun& r : runs) {
            a_max = std::max(a_max, align_up(tc_assemble_scratch(ctx, R, inst[r.i0].J, Fz[r.i0], r.n)));
            s_max = std::max(s_max, align_up(tc_synth_scratch(L0.U, L0.Vn, Fz[r.i0] * r.n)));
            if (det) w_max = std::max(w_max, tc_synth_wsum_bytes(Fz[r.i0] * r.n, Nx, Ny));
        }
        Carver probe(cv.base);
        probe.off = cv.off;
        probe.take(tc_synth_twiddle_bytes(L0.U, L0.Vn, Nx, Ny));
        void* a_scr = probe.take(a_max);
        void* s_scr = probe.take(s_max);
        void* w_scr = det ? probe.take(w_max) : nullptr;
        int* ctl = nullptr;
        size_t n_ctl = 0;                           // the control block starts the assembly scratch; sized for the largest run
        for (const SweepRun& r : runs) {
            size_t n = 0;
            tc_assemble_ctl(ctx, R, inst[r.i0].J, Fz[r.i0], r.n, a_scr, &ctl, &n);
            n_ctl = std::max(n_ctl, n);
        }
        bool clean = ctx->cache_on && ctx->clean_ctl == ctl && ctx->clean_ints >= n_ctl;
        bool zeroed = false;
        const Twiddles tw = run_twiddles(ctx, L0.dtype, L0.U, L0.Vn, L0.X, L0.Y, Nx, x, Ny, y, cv, clean ? nullptr : ctl,
                                         n_ctl, &zeroed);
        clean = clean || zeroed;
        if (!clean) {                               // cached twiddles but an unknown control block: clear all of it once
            cudaMemsetAsync(ctl, 0, n_ctl * sizeof(int), ctx->stream);
            clean = true;
        }
        // ints [0, clean_upto) of the control block hold zeros at this point of the stream.  Every run lays its per-CTA
        // timers, timeline ring, weight images and partial tiles out right behind ITS OWN counters, so after a run only its
        // own counters are known clean: a larger run that follows gets its counters cleared first.
        size_t clean_upto = n_ctl;
        for (const SweepRun& r : runs) {
            const int64_t i0 = r.i0, fz = Fz[i0];
            const int g = r.n;
            size_t n_run = 0;
            tc_assemble_ctl(ctx, R, inst[i0].J, fz, g, a_scr, &ctl, &n_run);
            if (n_run > clean_upto) cudaMemsetAsync(ctl, 0, n_run * sizeof(int), ctx->stream);
            clean_upto = n_run;
            TcFixup fix = {};
            int* sched = nullptr;
            int n_sched = 0;
            tc_synth_image_plan(L0.U, L0.Vn, Nx, Ny, s_scr, tw.a, &fix, &sched, &n_sched);
            // image padding: zeroed by the kernel unless an earlier launch left this very buffer in the same layout
            const int64_t planes = fz * 3 * g;
            fix.skip_zero = (ctx->cache_on || i0 > 0) && ctx->clean_img == s_scr && ctx->clean_img_U == L0.U &&
                            ctx->clean_img_Vn == L0.Vn && ctx->clean_img_planes >= planes;
            if (!fix.skip_zero) { ctx->clean_img = s_scr; ctx->clean_img_U = L0.U; ctx->clean_img_Vn = L0.Vn; ctx->clean_img_planes = planes; }
            launch_tc_assemble_group(ctx, g, inst + i0, fz, z + i0, fix, sched, n_sched, a_scr, clean);
            if (ctx->tc_error) return;
            clean = true;                               // the kernel leaves its control block zeroed (n_ctl ints were clean before)
            TcDetector td;
            if (det) {
                td.I = det->I ? det->I + i0 : nullptr;
                td.S = det->S ? det->S + i0 : nullptr;
                memcpy(td.win, det->win, sizeof(td.win));
                td.s_part = w_scr;
            }
            launch_tc_synth_group_images(ctx, L0.U, L0.Vn, fz, g, Nx, Ny, tw.a, det ? nullptr : E + i0, s4, s_scr,
                                         det ? &td : nullptr);
        }
        if (!ctx->cache_on) ctx->clean_img = nullptr;   // trusted across calls only under SCW_OPT_CACHE
        ctx->clean_ints = clean_upto;                   // what the LAST run left clean, not the largest run's block
        return;
    }
    // per-instance path: its P, assembly scratch and synthesis buffers overlay the grouped layout's control block and
    // spectrum images, so a later grouped sweep must not trust either (SCW_OPT_CACHE)
    ctx->clean_ctl = nullptr;
    ctx->clean_img = nullptr;
    const Twiddles tw = run_twiddles(ctx, L0.dtype, L0.U, L0.Vn, L0.X, L0.Y, Nx, x, Ny, y, cv);
    void* P = cv.take((size_t)R * fz_max * esize(L0.dtype));
    const size_t asm_off = cv.off;
    cv.take(asm_max);
    void* scratch = cv.take(synth_ws(ctx, L0.dtype, L0.U, L0.Vn, fz_max, Ny));
    void* E_tmp = det ? cv.take((size_t)fz_max * 3 * Nx * Ny * esize(L0.dtype)) : nullptr;   // general detector path
    int64_t planar[4];
    planar_strides(Nx, Ny, planar);
    for (int64_t i = 0; i < n_inst; ++i) {
        if (Fz[i] == 0) continue;
        Carver sub(cv.base ? cv.base + asm_off : nullptr);
        run_assemble(ctx, &inst[i], Fz[i], z[i], P, R, sub);
        if (det) {
            run_synth(ctx, tw, L0.dtype, L0.U, L0.Vn, Fz[i], P, R, Nx, Ny, E_tmp, planar, scratch);
            if (det->I) launch_intensity(ctx, L0.dtype, Fz[i], Ny, Nx, E_tmp, det->I[i], s4 + 1);
            if (det->S) launch_window_sum(ctx, L0.dtype, Fz[i], Ny, Nx, E_tmp, det->win, det->S[i]);
        } else {
            run_synth(ctx, tw, L0.dtype, L0.U, L0.Vn, Fz[i], P, R, Nx, Ny, E[i], s4, scratch);
        }
    }
}

static int32_t sweep_impl(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, const double* const* z,
                          int64_t Nx, const double* x, int64_t Ny, const double* y, void* const* E, const int64_t* strides,
                          const DetArgs* det, const char* who)
{
    if (int32_t s = check_ctx(ctx, true)) return s;
    int64_t fz_max = 0;
    size_t asm_max = 0;
    if (int32_t s = check_sweep(ctx, n_inst, inst, Fz, Nx, Ny, who, &fz_max, &asm_max)) return s;
    if (n_inst == 0 || fz_max == 0) return SCW_OK;
    if (int32_t s = check_grid(ctx, inst[0].dtype, inst[0].U, inst[0].Vn, inst[0].X, inst[0].Y, Nx, x, Ny, y, who)) return s;
    if (!z) return fail(ctx, SCW_ERR_NULL, "%s: z is required", who);
    if (!det && !E) return fail(ctx, SCW_ERR_NULL, "%s: the output array is required", who);
    if (det && !det->I && !det->S) return fail(ctx, SCW_ERR_NULL, "%s: at least one of I and S is required", who);
    if (det && (det->win[0] < 0 || det->win[1] > Nx || det->win[0] >= det->win[1] || det->win[2] < 0 || det->win[3] > Ny ||
                det->win[2] >= det->win[3]))
        return fail(ctx, SCW_ERR_SHAPE, "%s: window [%lld, %lld) x [%lld, %lld) is empty or outside the %lld x %lld grid", who,
                    (long long)det->win[0], (long long)det->win[1], (long long)det->win[2], (long long)det->win[3],
                    (long long)Nx, (long long)Ny);
    const size_t out_es = det ? esize(inst[0].dtype) / 2 : esize(inst[0].dtype);
    for (int64_t i = 0; i < n_inst; ++i) {
        if (Fz[i] == 0) continue;
        if (!z[i] || !aligned(z[i], 8)) return fail(ctx, SCW_ERR_NULL, "%s: z[%lld] is NULL or misaligned", who, (long long)i);
        void* outs[3] = {det ? nullptr : E[i], (det && det->I) ? det->I[i] : nullptr, (det && det->S) ? det->S[i] : nullptr};
        const bool wanted[3] = {!det, det && det->I, det && det->S};
        for (int k = 0; k < 3; ++k) {
            if (!wanted[k]) continue;
            if (!outs[k]) return fail(ctx, SCW_ERR_NULL, "%s: output[%lld] is NULL", who, (long long)i);
            if (!aligned(outs[k], out_es)) return fail(ctx, SCW_ERR_ALIGN, "%s: output[%lld] misaligned", who, (long long)i);
        }
    }
    int64_t s4[4];
    if (det) {                                         // (z, y, x) strides in s4[1..3]; the component slot is unused
        s4[0] = 0;
        if (strides) memcpy(s4 + 1, strides, 3 * sizeof(int64_t));
        else { s4[1] = Nx * Ny; s4[2] = Nx; s4[3] = 1; }
    } else if (strides) {
        memcpy(s4, strides, sizeof(s4));
    } else {
        planar_strides(Nx, Ny, s4);
    }
    for (int i = 0; i < 4; ++i)
        if (s4[i] < 0) return fail(ctx, SCW_ERR_SHAPE, "%s: negative stride", who);
    if (int32_t s = need_ws(ctx, sweep_need(ctx, n_inst, inst, Fz, fz_max, asm_max, Nx, Ny, det), who)) return s;
    Carver cv(ctx->ws);
    run_sweep(ctx, n_inst, inst, Fz, z, Nx, x, Ny, y, E, s4, fz_max, asm_max, cv, det);
    return check_launch(ctx, who);
}

int32_t scw_sweep_wavelengths(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz,
                              const double* const* z, int64_t Nx, const double* x, int64_t Ny, const double* y,
                              void* const* E, const int64_t* strides)
{
    return sweep_impl(ctx, n_inst, inst, Fz, z, Nx, x, Ny, y, E, strides, nullptr, "scw_sweep_wavelengths");
}

int32_t scw_sweep_detector(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz,
                           const double* const* z, int64_t Nx, const double* x, int64_t Ny, const double* y,
                           void* const* I, const int64_t* strides, const scw_window* window, void* const* S)
{
    DetArgs det;
    det.I = I;
    det.S = S;
    det.win[0] = window ? window->ix0 : 0;
    det.win[1] = window ? window->ix1 : Nx;
    det.win[2] = window ? window->iy0 : 0;
    det.win[3] = window ? window->iy1 : Ny;
    return sweep_impl(ctx, n_inst, inst, Fz, z, Nx, x, Ny, y, nullptr, strides, &det, "scw_sweep_detector");
}

int32_t scw_sweep_detector_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t Nx,
                                     int64_t Ny, size_t* bytes)
{
    return sweep_workspace_impl(ctx, n_inst, inst, Fz, Nx, Ny, bytes, true, "scw_sweep_detector_workspace");
}

int32_t scw_sweep_intensity(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz,
                            const double* const* z, int64_t Nx, const double* x, int64_t Ny, const double* y,
                            void* const* I, const int64_t* strides)
{
    if (ctx && !I) return fail(ctx, SCW_ERR_NULL, "scw_sweep_intensity: the output array is required");
    return scw_sweep_detector(ctx, n_inst, inst, Fz, z, Nx, x, Ny, y, I, strides, nullptr, nullptr);
}

int32_t scw_absorbance(scw_ctx* ctx, int32_t dtype, int64_t n, const void* S, const void* S0, const void* w, void* A,
                       void* band)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (dtype != SCW_C64 && dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "scw_absorbance: bad dtype %d", dtype);
    if (n < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_absorbance: n=%lld < 0", (long long)n);
    if (n == 0) return SCW_OK;
    if (!S || !S0 || (!A && !band)) return fail(ctx, SCW_ERR_NULL, "scw_absorbance: S, S0 and one of A, band are required");
    const size_t es = esize(dtype) / 2;
    if (!aligned(S, es) || !aligned(S0, es) || (w && !aligned(w, es)) || (A && !aligned(A, es)) || (band && !aligned(band, es)))
        return fail(ctx, SCW_ERR_ALIGN, "scw_absorbance: misaligned array");
    launch_absorbance(ctx, dtype, n, S, S0, w, A, band);
    return check_launch(ctx, "scw_absorbance");
}

int32_t scw_profile_assembly(scw_ctx* ctx, int32_t max_ctas, double* us, int32_t* n_ctas)
{
    if (!ctx || !us || !n_ctas) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    *n_ctas = 0;
    const int G = ctx->last_asm_G;
    if (G == 0 || !ctx->last_asm_ns) return SCW_OK;
    if (max_ctas < G) return fail(ctx, SCW_ERR_SHAPE, "scw_profile_assembly: room for %d CTAs, %d needed", max_ctas, G);
    std::vector<unsigned long long> ns((size_t)G * 4);
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpy(ns.data(), ctx->last_asm_ns, ns.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) {
        ctx->cuda_err = (int32_t)e;
        return fail(ctx, SCW_ERR_CUDA, "scw_profile_assembly: %s", cudaGetErrorString(e));
    }
    for (size_t i = 0; i < ns.size(); ++i) us[i] = (double)ns[i] * 1e-3;
    *n_ctas = G;
    return SCW_OK;
}

int32_t scw_profile_timeline(scw_ctx* ctx, int32_t max_n, uint64_t* exit_ns, int32_t* kernel_class, int32_t* n)
{
    if (!ctx || !exit_ns || !kernel_class || !n) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    *n = 0;
    if (!ctx->tl_last_ring || ctx->tl_seq == 0 || max_n < 1) return SCW_OK;
    unsigned long long ring[TL_RING];
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpy(ring, ctx->tl_last_ring, sizeof(ring), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) {
        ctx->cuda_err = (int32_t)e;
        return fail(ctx, SCW_ERR_CUDA, "scw_profile_timeline: %s", cudaGetErrorString(e));
    }
    int64_t cnt = ctx->tl_seq < TL_RING ? ctx->tl_seq : TL_RING;
    if (cnt > max_n) cnt = max_n;
    for (int64_t i = 0; i < cnt; ++i) {                 // oldest first
        const int slot = (int)((ctx->tl_seq - cnt + i) % TL_RING);
        exit_ns[i] = ring[slot];
        kernel_class[i] = ctx->tl_class[slot];
    }
    *n = (int32_t)cnt;
    return SCW_OK;
}

// ------------------------------------------------------------------------------------------
// Stream-K split calibration: the persistent CTAs of the tcgen05 assembly do not all stream from HBM at the same rate
// (the same groups of SMs are slower in every run, and how much depends on what the L2 is busy with when the kernel
// starts), so equal spans leave a tail.  Runs the given sweep as the caller will run it, reads the per-CTA durations of
// its assembly launch and sets every CTA's (= SM's) share proportional to its measured rate.
int32_t scw_calibrate(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, const double* const* z,
                      int64_t Nx, const double* x, int64_t Ny, const double* y, void* const* E, const int64_t* strides,
                      int32_t reps)
{
    if (!ctx) return SCW_ERR_NULL;
    if (reps < 1 || reps > 64) return fail(ctx, SCW_ERR_VALUE, "scw_calibrate: reps must be in [1, 64]");
    ctx->split_w.clear();
    std::vector<unsigned long long> ns;             // [G][4] per-CTA nanoseconds of one assembly launch, sized once G is known
    std::vector<double> best_w;                     // the split with the shortest assembly seen so far (empty = equal)
    double best_us = 1e30;
    const int rounds = 8;
    const double eta = 0.5;                          // 0.2 .. 0.7 and up to 24 rounds measured: no better
    for (int round = 0; round <= rounds; ++round) { // the last round only scores the last update
        std::vector<std::vector<double>> samples;
        std::vector<double> kernel_us;
        int G = 0;
        for (int r = 0; r <= reps; ++r) {           // the first sweep of a round is a warm-up
            ctx->last_asm_G = 0;
            if (int32_t s = sweep_impl(ctx, n_inst, inst, Fz, z, Nx, x, Ny, y, E, strides, nullptr, "scw_calibrate")) {
                ctx->split_w.clear();
                return s;
            }
            G = ctx->last_asm_G;
            if (G < 2) return SCW_OK;               // not on the tensor-core assembly: nothing to calibrate
            if (ns.size() < (size_t)G * 4) ns.resize((size_t)G * 4);
            cudaError_t e = cudaStreamSynchronize(ctx->stream);
            if (e == cudaSuccess)
                e = cudaMemcpy(ns.data(), ctx->last_asm_ns, (size_t)G * 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
            if (e != cudaSuccess) {
                ctx->cuda_err = (int32_t)e;
                ctx->split_w.clear();
                return fail(ctx, SCW_ERR_CUDA, "scw_calibrate: %s", cudaGetErrorString(e));
            }
            if (r == 0) continue;
            std::vector<double> rate(G);
            for (int c = 0; c < G; ++c)
                rate[c] = (double)(ctx->last_asm_span0[c + 1] - ctx->last_asm_span0[c]) /
                          (double)(ns[4 * c + 2] > ns[4 * c + 1] ? ns[4 * c + 2] - ns[4 * c + 1] : 1);      // main loop only
            samples.push_back(rate);
            double last_exit = 0.0;
            for (int c = 0; c < G; ++c) last_exit = std::max(last_exit, (double)ns[4 * c + 3] * 1e-3);
            kernel_us.push_back(last_exit);
        }
        std::sort(kernel_us.begin(), kernel_us.end());
        const double score = kernel_us[kernel_us.size() / 2];        // median over the repetitions of the slowest CTA's exit
        if (score < best_us) { best_us = score; best_w = ctx->split_w; }
        if (round == rounds) break;
        std::vector<double> w(G);
        double mean = 0.0;
        for (int c = 0; c < G; ++c) {               // median over the repetitions
            std::vector<double> v;
            for (auto& sm : samples) v.push_back(sm[c]);
            std::sort(v.begin(), v.end());
            w[c] = v[v.size() / 2];
            mean += w[c] / G;
        }
        // damped update towards the measured relative rate: a CTA's time is not proportional to its span (what one CTA
        // gives up, its neighbours on the same memory paths pick up), the undamped update oscillates
        const bool first = (int)ctx->split_w.size() != G;
        for (int c = 0; c < G; ++c) {
            const double old = first ? 1.0 : ctx->split_w[c];
            const double rel = w[c] / mean;                      // measured rate relative to the mean
            const double cur = old;                               // share it ran with
            w[c] = cur * (1.0 + eta * (rel / cur - 1.0));         // half way from the current share to the measured rate
            if (!(w[c] > 0.6)) w[c] = 0.6;                        // clipped: no span beyond ~1.5x the mean (bounds the partial-tile slots)
            if (w[c] > 1.5) w[c] = 1.5;
        }
        ctx->split_w = w;
    }
    ctx->split_w = best_w;
    return SCW_OK;
}

// ------------------------------------------------------------------------------------------
// Host-buffer variant: one staging area for the inputs and one for the output of an instance,
// reused in stream order.
static size_t host_stage_bytes(const scw_layer* L, int64_t Fz, int64_t Nx, int64_t Ny, size_t* e_bytes)
{
    const size_t es = esize(L->dtype);
    *e_bytes = align_up((size_t)Fz * 3 * Nx * Ny * es);
    return align_up((size_t)L->ldV * L->J * es) + align_up((size_t)L->J * es) + align_up((size_t)L->J * 16) +
           align_up((size_t)L->J) + align_up((size_t)Fz * 8);
}

static int32_t sweep_host_sizes(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t Nx,
                                int64_t Ny, const char* who, int64_t* fz_max, size_t* asm_max, size_t* in_max,
                                size_t* e_max)
{
    if (int32_t s = check_sweep(ctx, n_inst, inst, Fz, Nx, Ny, who, fz_max, asm_max)) return s;
    *in_max = *e_max = 0;
    for (int64_t i = 0; i < n_inst; ++i) {
        size_t eb = 0;
        const size_t ib = host_stage_bytes(&inst[i], Fz[i], Nx, Ny, &eb);
        if (ib > *in_max) *in_max = ib;
        if (eb > *e_max) *e_max = eb;
    }
    return SCW_OK;
}

int32_t scw_sweep_host_workspace(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz, int64_t Nx,
                                 int64_t Ny, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    int64_t fz_max = 0;
    size_t asm_max = 0, in_max = 0, e_max = 0;
    if (int32_t s = sweep_host_sizes(ctx, n_inst, inst, Fz, Nx, Ny, "scw_sweep_host_workspace", &fz_max, &asm_max,
                                     &in_max, &e_max)) return s;
    *bytes = n_inst ? align_up((size_t)Nx * 8) + align_up((size_t)Ny * 8) + 2 * in_max + 2 * e_max +
                          sweep_ws(ctx, &inst[0], fz_max, asm_max, Nx, Ny)
                    : 0;
    return SCW_OK;
}

int32_t scw_sweep_wavelengths_host(scw_ctx* ctx, int64_t n_inst, const scw_layer* inst, const int64_t* Fz,
                                   const double* const* z, int64_t Nx, const double* x, int64_t Ny, const double* y,
                                   void* const* E, int64_t* h2d_bytes, int64_t* d2h_bytes)
{
    if (int32_t s = check_ctx(ctx)) return s;
    int64_t fz_max = 0;
    size_t asm_max = 0, in_max = 0, e_max = 0;
    if (int32_t s = sweep_host_sizes(ctx, n_inst, inst, Fz, Nx, Ny, "scw_sweep_wavelengths_host", &fz_max, &asm_max,
                                     &in_max, &e_max)) return s;
    if (h2d_bytes) *h2d_bytes = 0;
    if (d2h_bytes) *d2h_bytes = 0;
    if (n_inst == 0 || fz_max == 0) return SCW_OK;
    if (int32_t s = check_grid(ctx, inst[0].dtype, inst[0].U, inst[0].Vn, inst[0].X, inst[0].Y, Nx, x, Ny, y,
                               "scw_sweep_wavelengths_host")) return s;
    if (!z || !E) return fail(ctx, SCW_ERR_NULL, "scw_sweep_wavelengths_host: z and E are required");
    for (int64_t i = 0; i < n_inst; ++i)
        if (Fz[i] > 0 && (!z[i] || !E[i])) return fail(ctx, SCW_ERR_NULL, "scw_sweep_wavelengths_host: z[i]/E[i] is NULL");
    const size_t total = align_up((size_t)Nx * 8) + align_up((size_t)Ny * 8) + 2 * in_max + 2 * e_max +
                         sweep_ws(ctx, &inst[0], fz_max, asm_max, Nx, Ny);
    if (int32_t s = need_ws(ctx, total, "scw_sweep_wavelengths_host")) return s;

    // copy streams and events are created on first use
    cudaError_t err = cudaSuccess;
    auto ok = [&](cudaError_t e) { if (err == cudaSuccess) err = e; };
    if (!ctx->h2d_stream) {
        ok(cudaStreamCreateWithFlags(&ctx->h2d_stream, cudaStreamNonBlocking));
        ok(cudaStreamCreateWithFlags(&ctx->d2h_stream, cudaStreamNonBlocking));
        ok(cudaEventCreateWithFlags(&ctx->ev_start, cudaEventDisableTiming));
        for (int b = 0; b < 2; ++b) {
            ok(cudaEventCreateWithFlags(&ctx->ev_in[b], cudaEventDisableTiming));
            ok(cudaEventCreateWithFlags(&ctx->ev_done[b], cudaEventDisableTiming));
            ok(cudaEventCreateWithFlags(&ctx->ev_out[b], cudaEventDisableTiming));
        }
    }

    Carver cv(ctx->ws);
    double* dx = (double*)cv.take((size_t)Nx * 8);
    double* dy = (double*)cv.take((size_t)Ny * 8);
    char* stage_in[2], *stage_e[2];
    for (int b = 0; b < 2; ++b) stage_in[b] = (char*)cv.take(in_max);
    for (int b = 0; b < 2; ++b) stage_e[b] = (char*)cv.take(e_max);
    const scw_layer& L0 = inst[0];
    const size_t es = esize(L0.dtype);
    const int64_t R = 3LL * L0.U * L0.Vn;
    int64_t up = 0, down = 0;
    auto h2d = [&](void* d, const void* h, size_t n, cudaStream_t st) {
        ok(cudaMemcpyAsync(d, h, n, cudaMemcpyHostToDevice, st));
        up += (int64_t)n;
    };
    h2d(dx, x, (size_t)Nx * 8, ctx->stream);
    h2d(dy, y, (size_t)Ny * 8, ctx->stream);
    const Twiddles tw = run_twiddles(ctx, L0.dtype, L0.U, L0.Vn, L0.X, L0.Y, Nx, dx, Ny, dy, cv);
    void* P = cv.take((size_t)R * fz_max * es);
    const size_t asm_off = cv.off;
    cv.take(asm_max);
    void* scratch = cv.take(synth_ws(ctx, L0.dtype, L0.U, L0.Vn, fz_max, Ny));
    int64_t s4[4];
    planar_strides(Nx, Ny, s4);
    // Pipeline over instances, two staging buffers each way: the host->device copy of instance i+1 and the device->host
    // copy of instance i-1 run on their own streams beside the kernels of instance i (full-duplex PCIe).  Everything is
    // ordered after the work already on the ctx stream (ev_start) and joined back into it at the end.
    ok(cudaEventRecord(ctx->ev_start, ctx->stream));
    ok(cudaStreamWaitEvent(ctx->h2d_stream, ctx->ev_start, 0));
    ok(cudaStreamWaitEvent(ctx->d2h_stream, ctx->ev_start, 0));
    int64_t used[2] = {0, 0};                          // how many instances went through buffer b so far
    int64_t k = 0;
    for (int64_t i = 0; i < n_inst && err == cudaSuccess; ++i) {
        if (Fz[i] == 0) continue;
        const int b = (int)(k++ & 1);
        scw_layer L = inst[i];
        Carver st(stage_in[b]);
        void* dV = st.take((size_t)L.ldV * L.J * es);
        void* dc = st.take((size_t)L.J * es);
        void* dg = st.take((size_t)L.J * 16);
        void* dd = st.take((size_t)L.J);
        void* dz = st.take((size_t)Fz[i] * 8);
        // inputs of buffer b may be overwritten once the kernels of its previous user are done
        if (used[b]) ok(cudaStreamWaitEvent(ctx->h2d_stream, ctx->ev_done[b], 0));
        h2d(dV, L.V, (size_t)L.ldV * L.J * es, ctx->h2d_stream);
        if (L.c) h2d(dc, L.c, (size_t)L.J * es, ctx->h2d_stream);
        h2d(dg, L.gamma, (size_t)L.J * 16, ctx->h2d_stream);
        if (L.dir) h2d(dd, L.dir, (size_t)L.J, ctx->h2d_stream);
        h2d(dz, z[i], (size_t)Fz[i] * 8, ctx->h2d_stream);
        ok(cudaEventRecord(ctx->ev_in[b], ctx->h2d_stream));
        L.V = dV;
        L.c = L.c ? dc : nullptr;
        L.gamma = (const double*)dg;
        L.dir = L.dir ? (const int8_t*)dd : nullptr;
        // kernels: need this instance's inputs, and the output buffer back from the copy of its previous user
        ok(cudaStreamWaitEvent(ctx->stream, ctx->ev_in[b], 0));
        if (used[b]) ok(cudaStreamWaitEvent(ctx->stream, ctx->ev_out[b], 0));
        Carver sub((char*)ctx->ws + asm_off);
        run_assemble(ctx, &L, Fz[i], (const double*)dz, P, R, sub);
        run_synth(ctx, tw, L0.dtype, L0.U, L0.Vn, Fz[i], P, R, Nx, Ny, stage_e[b], s4, scratch);
        ok(cudaEventRecord(ctx->ev_done[b], ctx->stream));
        const size_t eb = (size_t)Fz[i] * 3 * Nx * Ny * es;
        ok(cudaStreamWaitEvent(ctx->d2h_stream, ctx->ev_done[b], 0));
        ok(cudaMemcpyAsync(E[i], stage_e[b], eb, cudaMemcpyDeviceToHost, ctx->d2h_stream));
        ok(cudaEventRecord(ctx->ev_out[b], ctx->d2h_stream));
        down += (int64_t)eb;
        used[b]++;
    }
    for (int b = 0; b < 2; ++b)                        // join: results are complete in ctx-stream order
        if (used[b]) ok(cudaStreamWaitEvent(ctx->stream, ctx->ev_out[b], 0));
    if (err != cudaSuccess) {
        ctx->cuda_err = (int32_t)err;
        return fail(ctx, SCW_ERR_CUDA, "scw_sweep_wavelengths_host: %s", cudaGetErrorString(err));
    }
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return check_launch(ctx, "scw_sweep_wavelengths_host");
}

// ------------------------------------------------------------------------------------------
static int32_t check_modes(scw_ctx* ctx, const scw_modes* m, const char* who)
{
    if (!m) return fail(ctx, SCW_ERR_NULL, "%s: modes is NULL", who);
    if (m->struct_size != sizeof(scw_modes)) return fail(ctx, SCW_ERR_SHAPE, "%s: modes.struct_size mismatch", who);
    if (m->kind == SCW_MODES_DENSE) return check_layer(ctx, &m->layer, who);
    if (m->kind != SCW_MODES_PLANEWAVE) return fail(ctx, SCW_ERR_SHAPE, "%s: unknown modes.kind %d", who, m->kind);
    if (m->dtype != SCW_C64 && m->dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "%s: bad dtype %d", who, m->dtype);
    if (m->J <= 0) return fail(ctx, SCW_ERR_SHAPE, "%s: J must be positive", who);
    if (!finite_pos(m->lambda)) return fail(ctx, SCW_ERR_VALUE, "%s: lambda must be finite and > 0", who);
    if (!m->sx || !m->sy || !m->gamma || !m->zref || !m->p) return fail(ctx, SCW_ERR_NULL, "%s: sx, sy, gamma, zref, p are required", who);
    if (!aligned(m->sx, 8) || !aligned(m->sy, 8) || !aligned(m->gamma, 16) || !aligned(m->zref, 8) ||
        !aligned(m->p, esize(m->dtype)))
        return fail(ctx, SCW_ERR_ALIGN, "%s: mode arrays misaligned", who);
    return SCW_OK;
}

constexpr int64_t DENSE_CHUNK_MAX = 4096;   // points per pass of the dense point path
constexpr int64_t DENSE_CHUNK_MIN = 64;

static size_t dense_chunk_ws(const scw_ctx* ctx, const scw_layer* L, int64_t N, int64_t chunk)
{
    // the full chunks and the ragged last chunk split the mode index differently: take the larger need
    const int64_t R = 3LL * L->U * L->Vn;
    if (chunk > N) chunk = N;
    const int64_t tail = N % chunk;
    size_t a = assemble_ws(ctx, L, chunk);
    if (tail) { const size_t b = assemble_ws(ctx, L, tail); if (b > a) a = b; }
    return align_up((size_t)chunk * 8) + align_up((size_t)R * chunk * esize(L->dtype)) + a;
}

int32_t scw_points_workspace(scw_ctx* ctx, const scw_modes* modes, int64_t N, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    if (int32_t s = check_modes(ctx, modes, "scw_points_workspace")) return s;
    if (N < 0) return fail(ctx, SCW_ERR_SHAPE, "N < 0");
    if (N == 0) { *bytes = 0; return SCW_OK; }
    if (modes->kind == SCW_MODES_PLANEWAVE) *bytes = points_table_bytes(modes->dtype, modes->J);
    else *bytes = dense_chunk_ws(ctx, &modes->layer, N, DENSE_CHUNK_MAX);
    return SCW_OK;
}

int32_t scw_eval_points(scw_ctx* ctx, const scw_modes* modes, int64_t N, const double* r, void* E)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_modes(ctx, modes, "scw_eval_points")) return s;
    if (N < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_eval_points: N=%lld < 0", (long long)N);
    if (N == 0) return SCW_OK;
    if (!r || !E) return fail(ctx, SCW_ERR_NULL, "scw_eval_points: r and E are required");
    const int dtype = modes->kind == SCW_MODES_PLANEWAVE ? modes->dtype : modes->layer.dtype;
    if (!aligned(r, 8) || !aligned(E, esize(dtype))) return fail(ctx, SCW_ERR_ALIGN, "scw_eval_points: r/E misaligned");

    if (modes->kind == SCW_MODES_PLANEWAVE) {
        if (int32_t s = need_ws(ctx, points_table_bytes(dtype, modes->J), "scw_eval_points")) return s;
        launch_points_planewave(ctx, modes, N, r, E, ctx->ws);
        return check_launch(ctx, "scw_eval_points");
    }
    // dense: chunks of points sized to the registered workspace
    const scw_layer* L = &modes->layer;
    int64_t chunk = N < DENSE_CHUNK_MAX ? N : DENSE_CHUNK_MAX;
    while (chunk > DENSE_CHUNK_MIN && dense_chunk_ws(ctx, L, N, chunk) > ctx->ws_bytes) chunk = (chunk + 1) / 2;
    if (chunk > N) chunk = N;
    if (int32_t s = need_ws(ctx, dense_chunk_ws(ctx, L, N, chunk), "scw_eval_points")) return s;
    const int64_t R = 3LL * L->U * L->Vn;
    const size_t es = esize(dtype);
    for (int64_t p0 = 0; p0 < N; p0 += chunk) {
        const int64_t n = (N - p0) < chunk ? (N - p0) : chunk;
        Carver cv(ctx->ws);
        double* zc = (double*)cv.take((size_t)chunk * 8);
        void* P = cv.take((size_t)R * chunk * es);
        launch_extract_z(ctx, n, r + 3 * p0, zc);
        run_assemble(ctx, L, n, zc, P, R, cv);
        launch_point_synth(ctx, dtype, L->U, L->Vn, L->X, L->Y, n, r + 3 * p0, P, R, (char*)E + (size_t)p0 * 3 * es);
    }
    return check_launch(ctx, "scw_eval_points");
}

// No-allocation variant of the plane-wave point path: see include/scwatter.h.  Everything is checked before the first
// CUDA call that enqueues work; the table limit is a property of the library image, not of the ctx.
int32_t scw_eval_points_noalloc(scw_ctx* ctx, const scw_modes* modes, int64_t N, const double* r, void* E)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_modes(ctx, modes, "scw_eval_points_noalloc")) return s;
    if (modes->kind != SCW_MODES_PLANEWAVE)
        return fail(ctx, SCW_ERR_UNSUPPORTED, "scw_eval_points_noalloc: only SCW_MODES_PLANEWAVE tables (the dense kind needs "
                                              "scratch that grows with the problem: use scw_eval_points with a workspace)");
    if (N < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_eval_points_noalloc: N=%lld < 0", (long long)N);
    if (modes->dtype == SCW_C64 && modes->J > (int64_t)SCW_POINTS_NOALLOC_MAX_J)
        return fail(ctx, SCW_ERR_SHAPE, "scw_eval_points_noalloc: J=%lld plane waves exceed the built-in table of "
                                        "SCW_POINTS_NOALLOC_MAX_J=%d entries; split the table or use scw_eval_points",
                    (long long)modes->J, (int)SCW_POINTS_NOALLOC_MAX_J);
    if (N == 0) return SCW_OK;
    if (!r || !E) return fail(ctx, SCW_ERR_NULL, "scw_eval_points_noalloc: r and E are required");
    if (!aligned(r, 8) || !aligned(E, esize(modes->dtype)))
        return fail(ctx, SCW_ERR_ALIGN, "scw_eval_points_noalloc: r/E misaligned");
    const cudaError_t e = launch_points_planewave_noalloc(ctx, modes, N, r, E);
    if (e != cudaSuccess) {
        ctx->cuda_err = (int32_t)e;
        return fail(ctx, SCW_ERR_CUDA, "scw_eval_points_noalloc: %s", cudaGetErrorString(e));
    }
    return check_launch(ctx, "scw_eval_points_noalloc");
}

// ------------------------------------------------------------------------------------------
static int32_t check_exterior(scw_ctx* ctx, const scw_exterior* e, const char* who)
{
    if (!e) return fail(ctx, SCW_ERR_NULL, "%s: exterior descriptor is NULL", who);
    if (e->struct_size != sizeof(scw_exterior)) return fail(ctx, SCW_ERR_SHAPE, "%s: exterior.struct_size mismatch", who);
    if (e->dtype != SCW_C64 && e->dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "%s: bad dtype %d", who, e->dtype);
    if (e->side != SCW_SIDE_ABOVE && e->side != SCW_SIDE_BELOW) return fail(ctx, SCW_ERR_VALUE, "%s: bad side %d", who, e->side);
    if (e->U <= 0 || e->Vn <= 0 || e->U > MAX_FREQ || e->Vn > MAX_FREQ)
        return fail(ctx, SCW_ERR_SHAPE, "%s: U=%d Vn=%d out of range", who, e->U, e->Vn);
    if (!finite_pos(e->X) || !finite_pos(e->Y) || !finite_pos(e->lambda))
        return fail(ctx, SCW_ERR_VALUE, "%s: X, Y and lambda must be finite and > 0", who);
    if (!std::isfinite(e->n_re) || !std::isfinite(e->n_im) || !std::isfinite(e->z_face) ||
        (e->side == SCW_SIDE_ABOVE && e->p_inc && !std::isfinite(e->z_inc)))
        return fail(ctx, SCW_ERR_VALUE, "%s: n, z_face and z_inc must be finite", who);
    if (!e->p_face) return fail(ctx, SCW_ERR_NULL, "%s: p_face is required", who);
    if (e->side == SCW_SIDE_BELOW && e->p_inc) return fail(ctx, SCW_ERR_VALUE, "%s: p_inc is only defined above the sample", who);
    const size_t es = esize(e->dtype);
    if (!aligned(e->p_face, es) || (e->p_inc && !aligned(e->p_inc, es))) return fail(ctx, SCW_ERR_ALIGN, "%s: amplitudes misaligned", who);
    return SCW_OK;
}

int32_t scw_exterior_spectra(scw_ctx* ctx, const scw_exterior* ext, int64_t Fz, const double* z, void* P, int64_t ldP)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_exterior(ctx, ext, "scw_exterior_spectra")) return s;
    if (Fz < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_exterior_spectra: Fz=%lld < 0", (long long)Fz);
    if (Fz == 0) return SCW_OK;
    if (!z || !P) return fail(ctx, SCW_ERR_NULL, "scw_exterior_spectra: z and P are required");
    if (ldP < 3LL * ext->U * ext->Vn) return fail(ctx, SCW_ERR_SHAPE, "scw_exterior_spectra: ldP=%lld < 3*U*Vn", (long long)ldP);
    if (!aligned(z, 8) || !aligned(P, esize(ext->dtype))) return fail(ctx, SCW_ERR_ALIGN, "scw_exterior_spectra: z/P misaligned");
    launch_exterior_spectra(ctx, ext, Fz, z, P, ldP);
    return check_launch(ctx, "scw_exterior_spectra");
}

// eq. 9 + eq. 10 on a rectilinear grid in one call.  complex64 within the tensor-core synthesis' reach: twiddles (kept under
// SCW_OPT_CACHE), eq. 9 straight into the spectrum images, synthesis -- 3 launches, 2 cached, P never in memory; otherwise
// scw_exterior_spectra into the workspace followed by the synthesis of scw_synthesize_grid.
static size_t exterior_grid_ws(const scw_ctx* ctx, const scw_exterior* e, int64_t Fz, int64_t Nx, int64_t Ny)
{
    const size_t tw = twiddle_ws(ctx, e->dtype, e->U, e->Vn, Nx, Ny), sy = synth_ws(ctx, e->dtype, e->U, e->Vn, Fz, Ny);
    if (use_tc_synth(ctx, e->dtype, e->U, e->Vn)) return tw + sy;
    return tw + sy + align_up((size_t)3 * e->U * e->Vn * Fz * esize(e->dtype));
}

int32_t scw_exterior_grid_workspace(scw_ctx* ctx, const scw_exterior* ext, int64_t Fz, int64_t Nx, int64_t Ny, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    if (int32_t s = check_exterior(ctx, ext, "scw_exterior_grid_workspace")) return s;
    if (Fz < 0 || Nx <= 0 || Ny <= 0) return fail(ctx, SCW_ERR_SHAPE, "scw_exterior_grid_workspace: bad dimensions");
    *bytes = Fz ? exterior_grid_ws(ctx, ext, Fz, Nx, Ny) : 0;
    return SCW_OK;
}

int32_t scw_exterior_grid(scw_ctx* ctx, const scw_exterior* ext, int64_t Fz, const double* z, int64_t Nx, const double* x,
                          int64_t Ny, const double* y, void* E, const int64_t* strides)
{
    if (int32_t s = check_ctx(ctx, true)) return s;           // keeps the twiddle cache (same place in the workspace as a sweep's)
    ctx->clean_ctl = nullptr;                                  // ... but a sweep's control block and images may be overwritten
    ctx->clean_img = nullptr;
    if (int32_t s = check_exterior(ctx, ext, "scw_exterior_grid")) return s;
    if (int32_t s = check_grid(ctx, ext->dtype, ext->U, ext->Vn, ext->X, ext->Y, Nx, x, Ny, y, "scw_exterior_grid")) return s;
    if (Fz < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_exterior_grid: Fz=%lld < 0", (long long)Fz);
    if (Fz == 0) return SCW_OK;
    if (!z || !E) return fail(ctx, SCW_ERR_NULL, "scw_exterior_grid: z and E are required");
    if (!aligned(z, 8) || !aligned(E, esize(ext->dtype))) return fail(ctx, SCW_ERR_ALIGN, "scw_exterior_grid: z/E misaligned");
    int64_t s4[4];
    if (strides) memcpy(s4, strides, sizeof(s4)); else planar_strides(Nx, Ny, s4);
    for (int i = 0; i < 4; ++i)
        if (s4[i] < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_exterior_grid: negative stride");
    if (int32_t s = need_ws(ctx, exterior_grid_ws(ctx, ext, Fz, Nx, Ny), "scw_exterior_grid")) return s;
    Carver cv(ctx->ws);
    const Twiddles tw = run_twiddles(ctx, ext->dtype, ext->U, ext->Vn, ext->X, ext->Y, Nx, x, Ny, y, cv);
    void* scratch = cv.take(synth_ws(ctx, ext->dtype, ext->U, ext->Vn, Fz, Ny));
    if (tw.tc) {
        launch_tc_synth_exterior(ctx, ext, Fz, z, Nx, Ny, tw.a, E, s4, scratch);
    } else {
        const int64_t R = 3LL * ext->U * ext->Vn;
        void* P = cv.take((size_t)R * Fz * esize(ext->dtype));
        launch_exterior_spectra(ctx, ext, Fz, z, P, R);
        run_synth(ctx, tw, ext->dtype, ext->U, ext->Vn, Fz, P, R, Nx, Ny, E, s4, scratch);
    }
    return check_launch(ctx, "scw_exterior_grid");
}

int32_t scw_exterior_points_workspace(scw_ctx* ctx, const scw_exterior* ext, int64_t N, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    if (int32_t s = check_exterior(ctx, ext, "scw_exterior_points_workspace")) return s;
    if (N < 0) return fail(ctx, SCW_ERR_SHAPE, "N < 0");
    *bytes = N ? exterior_points_bytes(ext) : 0;
    return SCW_OK;
}

int32_t scw_exterior_points(scw_ctx* ctx, const scw_exterior* ext, int64_t N, const double* r, void* E)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_exterior(ctx, ext, "scw_exterior_points")) return s;
    if (N < 0) return fail(ctx, SCW_ERR_SHAPE, "scw_exterior_points: N=%lld < 0", (long long)N);
    if (N == 0) return SCW_OK;
    if (!r || !E) return fail(ctx, SCW_ERR_NULL, "scw_exterior_points: r and E are required");
    if (!aligned(r, 8) || !aligned(E, esize(ext->dtype))) return fail(ctx, SCW_ERR_ALIGN, "scw_exterior_points: r/E misaligned");
    if (int32_t s = need_ws(ctx, exterior_points_bytes(ext), "scw_exterior_points")) return s;
    launch_exterior_points(ctx, ext, N, r, E, ctx->ws);
    return check_launch(ctx, "scw_exterior_points");
}

// ------------------------------------------------------------------------------------------
static int32_t check_vbuild(scw_ctx* ctx, const scw_vbuild* vb, const char* who)
{
    if (!vb) return fail(ctx, SCW_ERR_NULL, "%s: descriptor is NULL", who);
    if (vb->struct_size != sizeof(scw_vbuild)) return fail(ctx, SCW_ERR_SHAPE, "%s: vbuild.struct_size mismatch", who);
    if (vb->dtype != SCW_C64 && vb->dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "%s: bad dtype %d", who, vb->dtype);
    if (vb->U <= 0 || vb->Vn <= 0 || vb->U > MAX_FREQ || vb->Vn > MAX_FREQ)
        return fail(ctx, SCW_ERR_SHAPE, "%s: U=%d Vn=%d out of range", who, vb->U, vb->Vn);
    if (vb->J <= 0) return fail(ctx, SCW_ERR_SHAPE, "%s: J must be positive", who);
    if (vb->ldQ < 4LL * vb->U * vb->Vn) return fail(ctx, SCW_ERR_SHAPE, "%s: ldQ=%lld < 4*U*Vn", who, (long long)vb->ldQ);
    if (!finite_pos(vb->X) || !finite_pos(vb->Y) || !finite_pos(vb->lambda))
        return fail(ctx, SCW_ERR_VALUE, "%s: X, Y and lambda must be finite and > 0", who);
    if (!vb->Q || !vb->psi) return fail(ctx, SCW_ERR_NULL, "%s: Q and psi are required", who);
    const size_t es = esize(vb->dtype);
    if (!aligned(vb->Q, es) || !aligned(vb->psi, es) || (vb->alpha && !aligned(vb->alpha, es)))
        return fail(ctx, SCW_ERR_ALIGN, "%s: Q/psi/alpha misaligned", who);
    return SCW_OK;
}

int32_t scw_build_V_workspace(scw_ctx* ctx, const scw_vbuild* vb, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    if (int32_t s = check_vbuild(ctx, vb, "scw_build_V_workspace")) return s;
    *bytes = vbuild_scratch(ctx, vb);
    return SCW_OK;
}

int32_t scw_build_V(scw_ctx* ctx, const scw_vbuild* vb, void* V, int64_t ldV)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_vbuild(ctx, vb, "scw_build_V")) return s;
    if (!V) return fail(ctx, SCW_ERR_NULL, "scw_build_V: V is required");
    if (ldV < 3LL * vb->U * vb->Vn) return fail(ctx, SCW_ERR_SHAPE, "scw_build_V: ldV=%lld < 3*U*Vn", (long long)ldV);
    if (!aligned(V, esize(vb->dtype))) return fail(ctx, SCW_ERR_ALIGN, "scw_build_V: V misaligned");
    if (int32_t s = need_ws(ctx, vbuild_scratch(ctx, vb), "scw_build_V")) return s;
    launch_vbuild(ctx, vb, V, ldV, ctx->ws);
    return check_launch(ctx, "scw_build_V");
}

// ------------------------------------------------------------------------------------------
static int32_t check_stack(scw_ctx* ctx, const scw_stack* st, const char* who)
{
    if (!st) return fail(ctx, SCW_ERR_NULL, "%s: descriptor is NULL", who);
    if (st->struct_size != sizeof(scw_stack)) return fail(ctx, SCW_ERR_SHAPE, "%s: stack.struct_size mismatch", who);
    if (st->dtype != SCW_C64 && st->dtype != SCW_C128) return fail(ctx, SCW_ERR_DTYPE, "%s: bad dtype %d", who, st->dtype);
    if (st->n_layers <= 0 || st->n <= 0) return fail(ctx, SCW_ERR_SHAPE, "%s: n_layers and n must be positive", who);
    if (st->ldQ < st->n) return fail(ctx, SCW_ERR_SHAPE, "%s: ldQ=%lld < n=%lld", who, (long long)st->ldQ, (long long)st->n);
    if (!finite_pos(st->lambda)) return fail(ctx, SCW_ERR_VALUE, "%s: lambda must be finite and > 0", who);
    if (!st->z_if || !st->Q || !st->gamma) return fail(ctx, SCW_ERR_NULL, "%s: z_if, Q and gamma are required", who);
    for (int l = 0; l <= st->n_layers; ++l)
        if (!std::isfinite(st->z_if[l]) || (l > 0 && st->z_if[l] < st->z_if[l - 1]))
            return fail(ctx, SCW_ERR_VALUE, "%s: interfaces must be finite and non-decreasing", who);
    const size_t es = esize(st->dtype);
    for (int l = 0; l < st->n_layers; ++l) {
        if (!st->Q[l] || !st->gamma[l]) return fail(ctx, SCW_ERR_NULL, "%s: Q[%d] / gamma[%d] is NULL", who, l, l);
        if (!aligned(st->Q[l], es) || !aligned(st->gamma[l], 16)) return fail(ctx, SCW_ERR_ALIGN, "%s: Q[%d] / gamma[%d] misaligned", who, l, l);
    }
    if (!alpha_supported(ctx, st->n))
        return fail(ctx, SCW_ERR_UNSUPPORTED, "%s: n=%lld beyond the LU's limit on this device", who, (long long)st->n);
    return SCW_OK;
}

int32_t scw_propagate_alpha_workspace(scw_ctx* ctx, const scw_stack* st, size_t* bytes)
{
    if (!ctx || !bytes) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    if (int32_t s = check_stack(ctx, st, "scw_propagate_alpha_workspace")) return s;
    *bytes = alpha_scratch(ctx, st->n);
    return SCW_OK;
}

int32_t scw_propagate_alpha(scw_ctx* ctx, const scw_stack* st, const void* r0, void* const* alpha, void* rL)
{
    if (int32_t s = check_ctx(ctx)) return s;
    if (int32_t s = check_stack(ctx, st, "scw_propagate_alpha")) return s;
    if (!r0 || !alpha) return fail(ctx, SCW_ERR_NULL, "scw_propagate_alpha: r0 and alpha are required");
    const size_t es = esize(st->dtype);
    if (!aligned(r0, es) || (rL && !aligned(rL, es))) return fail(ctx, SCW_ERR_ALIGN, "scw_propagate_alpha: r0 / rL misaligned");
    for (int l = 0; l < st->n_layers; ++l)
        if (!alpha[l] || !aligned(alpha[l], es)) return fail(ctx, SCW_ERR_NULL, "scw_propagate_alpha: alpha[%d] is NULL or misaligned", l);
    if (int32_t s = need_ws(ctx, alpha_scratch(ctx, st->n), "scw_propagate_alpha")) return s;
    launch_propagate_alpha(ctx, st, r0, alpha, rL, ctx->ws);
    return check_launch(ctx, "scw_propagate_alpha");
}

}  // extern "C"
