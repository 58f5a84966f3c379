// Point path of libscw (step a-5 / a-6): direct plane-wave sum at scattered points
//   E(r_p) = sum_j p_j exp(i k [s_xj x_p + s_yj y_p + gamma_j (z_p - zref_j)])
// (discrete eq. 3; eq. 9-10; any s_m).
//
// complex64 kernel: the phase in turns is accumulated by three fp64 FMAs onto the constant
// 1.5*2^20, which leaves frac(phase) * 2^32 in the low word of the double (fp64 range reduction
// without a rint); sin/cos/exp2 run on the MUFU pipe, the three complex MACs as packed fp32
// FMAs (FFMA2).  Every thread carries PPT points so that one broadcast read of a mode entry
// from shared memory feeds PPT term evaluations.
// Domain: the magic-constant reduction is exact only while |phase| < 2^19 turns.  Phases are therefore taken relative
// to the first point r_0 of the call (the per-mode part a_j . r_0 is reduced with rint in fp64 by the table kernel
// and folded into c0), so the limit applies to the EXTENT of the point cloud, not to its distance from the origin;
// a block that holds a point whose bound |a|_max . |r - r_0| reaches 2^19 turns takes a second loop that reduces every
// term with rint first (any finite coordinate is then evaluated correctly, at ~1.3x the cost for that block).
#include <mutex>

#include "scw_internal.h"

namespace scw {

constexpr double PW_MAGIC = 1572864.0;             // 1.5 * 2^20: ulp = 2^-32 turn
constexpr double PW_FAST_LIMIT = 524000.0;         // < 2^19 - 1: |phase relative to r_0| up to here takes the fast loop
#ifndef SCW_PW_PPT
#define SCW_PW_PPT 4
#endif
#ifndef SCW_PW_MINBLOCKS
#define SCW_PW_MINBLOCKS 1
#endif
constexpr int PW_THREADS = 128;
constexpr int PW_PPT = SCW_PW_PPT;                 // points per thread
constexpr int PW_CHUNK = 256;                      // modes staged per shared-memory chunk

struct __align__(16) PwMode {                      // 96 bytes
    double ax, ay, az, c0;                         // turns per unit length; c0 = MAGIC + frac(a . r_0 - az*zref)
    float nkap, ke0, pad0, pad1;                   // log2-amplitude = nkap*(z - z_0) + ke0
    float prr[3][2];                               // (p_re, p_re) per component
    float pii[3][2];                               // (p_im, p_im) per component
};
static_assert(sizeof(PwMode) == 96, "PwMode layout");

// Table header (first 256 bytes of the table buffer, zeroed before k_points_table): max_j |ax|, |ay|, |az| as the bit
// patterns of non-negative doubles (monotone under unsigned compare, so atomicMax works).
struct PwHeader { unsigned long long max_a[3]; };
constexpr size_t PW_HEADER_BYTES = 256;

template <typename T2>
__global__ void k_points_table(int64_t J, double inv_lambda, const double* __restrict__ sx,
                               const double* __restrict__ sy, const double2* __restrict__ gamma,
                               const double* __restrict__ zref, const T2* __restrict__ p,
                               const double* __restrict__ r, PwHeader* __restrict__ hdr, PwMode* __restrict__ table)
{
    // every lane stays alive for the warp reduction at the end: lanes past J redo mode J - 1 and only skip the store
    // (their maxima equal that mode's, so the reduction is unchanged)
    const int64_t j_raw = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = j_raw < J;
    const int64_t j = live ? j_raw : J - 1;
    const double x0 = r[0], y0 = r[1], z0 = r[2];                 // phase origin: the first point of the call
    const double2 g = gamma[j];
    PwMode m;
    m.ax = sx[j] * inv_lambda;
    m.ay = sy[j] * inv_lambda;
    m.az = g.x * inv_lambda;
    // phase of the mode at r_0 in turns, each product reduced on its own (|a x_0| may be 1e5 turns and more)
    double t0 = m.ax * x0;
    t0 -= rint(t0);
    double t1 = m.ay * y0;
    t1 -= rint(t1);
    double t2 = m.az * (z0 - zref[j]);
    t2 -= rint(t2);
    double f = t0 + t1 + t2;
    f -= rint(f);
    m.c0 = PW_MAGIC + f;
    const double kap = 6.283185307179586476925 * 1.4426950408889634074 * g.y * inv_lambda;
    m.nkap = (float)(-kap);
    m.ke0 = (float)(kap * (zref[j] - z0));
    m.pad0 = m.pad1 = 0.f;
    for (int c = 0; c < 3; ++c) {
        const T2 v = p[3 * j + c];
        m.prr[c][0] = m.prr[c][1] = (float)v.x;
        m.pii[c][0] = m.pii[c][1] = (float)v.y;
    }
    if (live) table[j] = m;
    // per-axis maxima for the domain check of the fast loop: one atomic per warp and axis
    double a3[3] = {fabs(m.ax), fabs(m.ay), fabs(m.az)};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        unsigned long long b = (unsigned long long)__double_as_longlong(a3[k]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
            b = other > b ? other : b;
        }
        if ((threadIdx.x & 31) == 0) atomicMax(&hdr->max_a[k], b);
    }
}

__device__ __forceinline__ float ex2_approx(float x)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// One chunk of modes against the PPT points of the thread.  REDUCE: every term is first reduced with rint (phases of
// any size); otherwise the three FMAs land directly on the magic constant (|phase| < 2^19 turns).
template <bool REDUCE>
__device__ __forceinline__ void pw_chunk(const PwMode* __restrict__ sm, int nj, const double (&x)[PW_PPT],
                                         const double (&y)[PW_PPT], const double (&z)[PW_PPT], const float (&z32)[PW_PPT],
                                         float2 (&A)[PW_PPT][3], float2 (&B)[PW_PPT][3])
{
#pragma unroll 1
    for (int jj = 0; jj < nj; ++jj) {
        const double2 a01 = *reinterpret_cast<const double2*>(&sm[jj].ax);
        const double2 a23 = *reinterpret_cast<const double2*>(&sm[jj].az);
        const float4 kk = *reinterpret_cast<const float4*>(&sm[jj].nkap);
        const float4 p0 = *reinterpret_cast<const float4*>(&sm[jj].prr[0][0]);
        const float4 p1 = *reinterpret_cast<const float4*>(&sm[jj].prr[2][0]);
        const float4 p2 = *reinterpret_cast<const float4*>(&sm[jj].pii[1][0]);
        const float2 prr0 = make_float2(p0.x, p0.y), prr1 = make_float2(p0.z, p0.w);
        const float2 prr2 = make_float2(p1.x, p1.y), pii0 = make_float2(p1.z, p1.w);
        const float2 pii1 = make_float2(p2.x, p2.y), pii2 = make_float2(p2.z, p2.w);
#pragma unroll
        for (int q = 0; q < PW_PPT; ++q) {
            double t;
            if (REDUCE) {
                t = fma(a01.x, x[q], fma(a01.y, y[q], fma(a23.x, z[q], a23.y - PW_MAGIC)));
                t = (t - rint(t)) + PW_MAGIC;
            } else {
                t = fma(a01.x, x[q], fma(a01.y, y[q], fma(a23.x, z[q], a23.y)));
            }
            const int ph = __double2loint(t);                 // frac(turns) * 2^32, signed
            const float ang = __int2float_rn(ph) * 1.4629180792671596e-9f;   // 2 pi / 2^32
            const float sn = __sinf(ang), cs = __cosf(ang);
            const float amp = ex2_approx(fmaf(kk.x, z32[q], kk.y));
            const float2 w = make_float2(amp * cs, amp * sn);
            A[q][0] = __ffma2_rn(prr0, w, A[q][0]);
            B[q][0] = __ffma2_rn(pii0, w, B[q][0]);
            A[q][1] = __ffma2_rn(prr1, w, A[q][1]);
            B[q][1] = __ffma2_rn(pii1, w, B[q][1]);
            A[q][2] = __ffma2_rn(prr2, w, A[q][2]);
            B[q][2] = __ffma2_rn(pii2, w, B[q][2]);
        }
    }
}

__global__ void __launch_bounds__(PW_THREADS, SCW_PW_MINBLOCKS)
k_points_pw_c64(int64_t J, int64_t N, const double* __restrict__ r, const PwHeader* __restrict__ hdr,
                const PwMode* __restrict__ table, float2* __restrict__ E)
{
    __shared__ PwMode sm[PW_CHUNK];
    const int tid = threadIdx.x;
    const int64_t base = (int64_t)blockIdx.x * (PW_THREADS * PW_PPT);
    const double x0 = r[0], y0 = r[1], z0 = r[2];
    const double max_ax = __longlong_as_double((long long)hdr->max_a[0]);
    const double max_ay = __longlong_as_double((long long)hdr->max_a[1]);
    const double max_az = __longlong_as_double((long long)hdr->max_a[2]);

    double x[PW_PPT], y[PW_PPT], z[PW_PPT];
    float z32[PW_PPT];
    float2 A[PW_PPT][3], B[PW_PPT][3];
    bool far = false;
#pragma unroll
    for (int q = 0; q < PW_PPT; ++q) {
        int64_t ip = base + q * PW_THREADS + tid;
        if (ip >= N) ip = N - 1;
        x[q] = r[3 * ip + 0] - x0;                  // coordinates relative to the first point
        y[q] = r[3 * ip + 1] - y0;
        z[q] = r[3 * ip + 2] - z0;
        z32[q] = (float)z[q];
        const double bound = fabs(x[q]) * max_ax + fabs(y[q]) * max_ay + fabs(z[q]) * max_az;
        far = far || !(bound < PW_FAST_LIMIT);      // NaN / inf coordinates go to the reducing loop too
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            A[q][c] = make_float2(0.f, 0.f);
            B[q][c] = make_float2(0.f, 0.f);
        }
    }
    const bool reduce = __syncthreads_or(far ? 1 : 0) != 0;    // block-uniform choice of the loop

    for (int64_t j0 = 0; j0 < J; j0 += PW_CHUNK) {
        const int nj = (int)min((int64_t)PW_CHUNK, J - j0);
        __syncthreads();
        {
            const uint4* __restrict__ src = reinterpret_cast<const uint4*>(table + j0);
            uint4* dst = reinterpret_cast<uint4*>(sm);
            const int n16 = nj * (int)(sizeof(PwMode) / 16);
            for (int i = tid; i < n16; i += PW_THREADS) dst[i] = src[i];
        }
        __syncthreads();
        if (reduce) pw_chunk<true>(sm, nj, x, y, z, z32, A, B);
        else pw_chunk<false>(sm, nj, x, y, z, z32, A, B);
    }
    // E = (A.x - B.y, A.y + B.x): sum p_re*w + i p_im*w
#pragma unroll
    for (int q = 0; q < PW_PPT; ++q) {
        const int64_t ip = base + q * PW_THREADS + tid;
        if (ip < N) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
                E[3 * ip + c] = make_float2(A[q][c].x - B[q][c].y, A[q][c].y + B[q][c].x);
        }
    }
}

// complex128 output: everything in fp64 (reduction by rint, sincospi, exp).
__global__ void __launch_bounds__(128)
k_points_pw_c128(int64_t J, int64_t N, double inv_lambda, const double* __restrict__ r,
                 const double* __restrict__ sx, const double* __restrict__ sy,
                 const double2* __restrict__ gamma, const double* __restrict__ zref,
                 const double2* __restrict__ p, double2* __restrict__ E)
{
    const int64_t ip = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= N) return;
    const double x = r[3 * ip], y = r[3 * ip + 1], z = r[3 * ip + 2];
    double er[3] = {0, 0, 0}, ei[3] = {0, 0, 0};
    for (int64_t j = 0; j < J; ++j) {
        const double2 g = gamma[j];
        const double dz = z - zref[j];
        double t = (sx[j] * x + sy[j] * y + g.x * dz) * inv_lambda;
        t -= rint(t);
        double s, c;
        sincospi(2.0 * t, &s, &c);
        const double a = exp(-6.283185307179586476925 * g.y * dz * inv_lambda);
        const double wr = a * c, wi = a * s;
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
            const double2 pv = p[3 * j + cc];
            er[cc] += pv.x * wr - pv.y * wi;
            ei[cc] += pv.x * wi + pv.y * wr;
        }
    }
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) E[3 * ip + cc] = make_double2(er[cc], ei[cc]);
}

size_t points_table_bytes(int dtype, int64_t J)
{
    return dtype == SCW_C64 ? PW_HEADER_BYTES + align_up((size_t)J * sizeof(PwMode)) : 0;
}

void launch_points_planewave(scw_ctx* ctx, const scw_modes* m, int64_t N, const double* r, void* E,
                             void* table)
{
    if (m->dtype == SCW_C64) {
        PwHeader* hdr = static_cast<PwHeader*>(table);
        PwMode* modes = reinterpret_cast<PwMode*>(static_cast<char*>(table) + PW_HEADER_BYTES);
        cudaMemsetAsync(hdr, 0, sizeof(PwHeader), ctx->stream);
        {
            KernelScope ks(ctx, KC_POINTS_TABLE);
            k_points_table<float2><<<(unsigned)((m->J + 127) / 128), 128, 0, ctx->stream>>>(
                m->J, 1.0 / m->lambda, m->sx, m->sy, (const double2*)m->gamma, m->zref, (const float2*)m->p, r, hdr, modes);
        }
        const int64_t per_block = PW_THREADS * PW_PPT;
        KernelScope ks(ctx, KC_POINTS);
        k_points_pw_c64<<<(unsigned)((N + per_block - 1) / per_block), PW_THREADS, 0, ctx->stream>>>(
            m->J, N, r, hdr, modes, (float2*)E);
    } else {
        KernelScope ks(ctx, KC_POINTS);
        k_points_pw_c128<<<(unsigned)((N + 127) / 128), 128, 0, ctx->stream>>>(
            m->J, N, 1.0 / m->lambda, r, m->sx, m->sy, (const double2*)m->gamma, m->zref,
            (const double2*)m->p, (double2*)E);
    }
}

// ------------------------------------------------------------------------------------------
// scw_eval_points_noalloc (include/scwatter.h): the same two complex64 kernels with the mode table in an array that is
// part of the library image instead of the caller's workspace, for callers that cannot allocate device memory.
//
// g_pw_noalloc is a __device__ variable.  Inside kernels of THIS file its name is the array; in host code the name only
// stands for the symbol (taking its address on the host gives a host address that no kernel may be handed), so the host
// asks the runtime where the current device keeps it -- cudaGetSymbolAddress -- and passes that pointer to the kernels
// like any other scratch buffer.  Every device has its own copy at its own address: the look-up is done once per device,
// with that device current, and remembered in g_pw_noalloc_addr.
constexpr size_t PW_NOALLOC_BYTES = PW_HEADER_BYTES + (size_t)SCW_POINTS_NOALLOC_MAX_J * sizeof(PwMode);
static __device__ __align__(256) unsigned char g_pw_noalloc[PW_NOALLOC_BYTES];

constexpr int PW_NOALLOC_MAX_DEV = 64;              // devices whose address is remembered; beyond: looked up every call
static std::mutex g_pw_noalloc_mu;
static void* g_pw_noalloc_addr[PW_NOALLOC_MAX_DEV]; // device address of g_pw_noalloc on device d, NULL = not looked up yet

// Device address of the built-in table on `device`, which the caller has made current.  No allocation.
static cudaError_t pw_noalloc_scratch(int device, void** out)
{
    std::lock_guard<std::mutex> lk(g_pw_noalloc_mu);
    const bool slot = device >= 0 && device < PW_NOALLOC_MAX_DEV;
    if (slot && g_pw_noalloc_addr[device]) {
        *out = g_pw_noalloc_addr[device];
        return cudaSuccess;
    }
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_pw_noalloc);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (slot) g_pw_noalloc_addr[device] = p;
    *out = p;
    return cudaSuccess;
}

// Enqueues header clear + table + sum on the ctx stream (SCW_C64, J <= SCW_POINTS_NOALLOC_MAX_J, checked by the entry
// point).  Launch accounting without KernelScope: its profiling branch creates CUDA events, which this path must not.
cudaError_t launch_points_planewave_noalloc(scw_ctx* ctx, const scw_modes* m, int64_t N, const double* r, void* E)
{
    if (m->dtype != SCW_C64) {                      // complex128: no table at all, the plain kernel
        ctx->launches++;
        ctx->last_classes |= 1ull << KC_POINTS;
        k_points_pw_c128<<<(unsigned)((N + 127) / 128), 128, 0, ctx->stream>>>(
            m->J, N, 1.0 / m->lambda, r, m->sx, m->sy, (const double2*)m->gamma, m->zref, (const double2*)m->p, (double2*)E);
        return cudaSuccess;
    }
    void* scratch = nullptr;
    if (cudaError_t e = pw_noalloc_scratch(ctx->device, &scratch)) return e;
    PwHeader* hdr = static_cast<PwHeader*>(scratch);
    PwMode* modes = reinterpret_cast<PwMode*>(static_cast<char*>(scratch) + PW_HEADER_BYTES);
    // the array still holds the previous call's maxima and table: the maxima must start at zero (atomicMax), the J
    // entries the sum reads are all rewritten by the table kernel
    if (cudaError_t e = cudaMemsetAsync(hdr, 0, sizeof(PwHeader), ctx->stream)) return e;
    ctx->launches += 2;
    ctx->last_classes |= (1ull << KC_POINTS_TABLE) | (1ull << KC_POINTS);
    k_points_table<float2><<<(unsigned)((m->J + 127) / 128), 128, 0, ctx->stream>>>(
        m->J, 1.0 / m->lambda, m->sx, m->sy, (const double2*)m->gamma, m->zref, (const float2*)m->p, r, hdr, modes);
    const int64_t per_block = PW_THREADS * PW_PPT;
    k_points_pw_c64<<<(unsigned)((N + per_block - 1) / per_block), PW_THREADS, 0, ctx->stream>>>(
        m->J, N, r, hdr, modes, (float2*)E);
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------
// a-6 helper: per-point Fourier synthesis of a spectrum column (eq. 10 at one point):
//   E[p,comp] = sum_{u,v} P[comp*M + v*U + u, p] exp(i 2 pi u x_p / X) exp(i 2 pi v y_p / Y)
// One warp per point; twiddles in fp64 -> T.
template <typename T, typename T2>
__global__ void __launch_bounds__(128)
k_point_synth(int U, int Vn, double invX, double invY, int64_t n, const double* __restrict__ r,
              const T2* __restrict__ P, int64_t ldP, T2* __restrict__ E)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    T2* fx = reinterpret_cast<T2*>(smem_raw) + (size_t)warp * (U + Vn);
    T2* fy = fx + U;
    const int64_t ip = (int64_t)blockIdx.x * 4 + warp;
    if (ip >= n) return;
    const double x = r[3 * ip] * invX, y = r[3 * ip + 1] * invY;
    for (int f = lane; f < U + Vn; f += 32) {
        double t = f < U ? (double)(f - U / 2) * x : (double)(f - U - Vn / 2) * y;
        t -= rint(t);
        double s, c;
        sincospi(2.0 * t, &s, &c);
        T2 w; w.x = (T)c; w.y = (T)s;
        fx[f] = w;
    }
    __syncwarp();
    const int64_t M = (int64_t)U * Vn;
    for (int comp = 0; comp < 3; ++comp) {
        const T2* __restrict__ col = P + ip * ldP + comp * M;
        T ar = 0, ai = 0;
        for (int64_t m = lane; m < M; m += 32) {
            const int v = (int)(m / U), u = (int)(m - (int64_t)v * U);
            const T2 a = fx[u], b = fy[v], pv = col[m];
            const T tr = a.x * b.x - a.y * b.y, ti = a.x * b.y + a.y * b.x;
            ar += pv.x * tr - pv.y * ti;
            ai += pv.x * ti + pv.y * tr;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            ar += __shfl_xor_sync(0xffffffffu, ar, o);
            ai += __shfl_xor_sync(0xffffffffu, ai, o);
        }
        if (lane == 0) { T2 e; e.x = ar; e.y = ai; E[3 * ip + comp] = e; }
    }
}

void launch_point_synth(scw_ctx* ctx, int dtype, int U, int Vn, double X, double Y, int64_t n,
                        const double* r, const void* P, int64_t ldP, void* E)
{
    const unsigned blocks = (unsigned)((n + 3) / 4);
    KernelScope ks(ctx, KC_POINT_SYNTH);
    if (dtype == SCW_C64)
        k_point_synth<float, float2><<<blocks, 128, 4 * (U + Vn) * sizeof(float2), ctx->stream>>>(
            U, Vn, 1.0 / X, 1.0 / Y, n, r, (const float2*)P, ldP, (float2*)E);
    else
        k_point_synth<double, double2><<<blocks, 128, 4 * (U + Vn) * sizeof(double2), ctx->stream>>>(
            U, Vn, 1.0 / X, 1.0 / Y, n, r, (const double2*)P, ldP, (double2*)E);
}

__global__ void k_extract_z(int64_t n, const double* __restrict__ r, double* __restrict__ z)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) z[i] = r[3 * i + 2];
}

void launch_extract_z(scw_ctx* ctx, int64_t n, const double* r, double* z)
{
    KernelScope ks(ctx, KC_MISC);
    k_extract_z<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(n, r, z);
}

}  // namespace scw
