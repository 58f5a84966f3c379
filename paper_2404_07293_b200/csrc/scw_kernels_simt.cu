// CUDA-core (SIMT) kernels of libscw: mode weights, twiddle tables, and the general-shape
// fallbacks for the two contractions (fp32 FMA for complex64, fp64 DFMA for complex128).
// Citations are PAPER.md line numbers.
#include "scw_internal.h"

namespace scw {

template <typename T> struct C2;
template <> struct C2<float> { using type = float2; };
template <> struct C2<double> { using type = double2; };

template <typename T2, typename T>
__device__ __forceinline__ T2 mk2(T a, T b) { T2 r; r.x = a; r.y = b; return r; }

// acc += a * b (complex)
template <typename T2>
__device__ __forceinline__ void cfma(T2& acc, const T2 a, const T2 b)
{
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}

__device__ __forceinline__ int mode_dir(const int8_t* dir, const double2 g, int64_t j)
{
    if (dir) return dir[j] > 0 ? 1 : -1;
    return (g.y > 0.0 || (g.y == 0.0 && g.x >= 0.0)) ? 1 : -1;
}

// ------------------------------------------------------------------------------------------
// a-1 mode weights: W[j,i] = c_j G(gamma_j, zref_j, z_i)   (eq. 7; eq. 30, :324-330)
// Always evaluated in fp64 (phase in turns, exact reduction, sincospi), rounded to T at the end.
template <typename T>
__global__ void k_mode_weights(int64_t J, int64_t Fz, double inv_lambda, double z_lo, double z_hi,
                               const typename C2<T>::type* __restrict__ c,
                               const double2* __restrict__ gamma, const int8_t* __restrict__ dir,
                               const double* __restrict__ z, typename C2<T>::type* __restrict__ W)
{
    using T2 = typename C2<T>::type;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= J * Fz) return;
    const int64_t j = idx / Fz, i = idx - j * Fz;
    const double2 g = gamma[j];
    const double dz = z[i] - (mode_dir(dir, g, j) > 0 ? z_lo : z_hi);
    double t = g.x * dz * inv_lambda;
    t -= rint(t);
    double s, co;
    sincospi(2.0 * t, &s, &co);
    const double a = exp(-6.283185307179586476925 * g.y * dz * inv_lambda);
    double cr = 1.0, ci = 0.0;
    if (c) { cr = (double)c[j].x; ci = (double)c[j].y; }
    const double wr = a * co, wi = a * s;
    W[idx] = mk2<T2, T>((T)(cr * wr - ci * wi), (T)(cr * wi + ci * wr));
}

void launch_mode_weights(scw_ctx* ctx, int dtype, int64_t J, int64_t Fz, double lambda, double z_lo,
                         double z_hi, const void* c, const double* gamma, const int8_t* dir,
                         const double* z, void* W)
{
    const int64_t n = J * Fz;
    const int threads = 256;
    const unsigned blocks = (unsigned)((n + threads - 1) / threads);
    KernelScope ks(ctx, KC_WEIGHTS);
    if (dtype == SCW_C64)
        k_mode_weights<float><<<blocks, threads, 0, ctx->stream>>>(
            J, Fz, 1.0 / lambda, z_lo, z_hi, (const float2*)c, (const double2*)gamma, dir, z, (float2*)W);
    else
        k_mode_weights<double><<<blocks, threads, 0, ctx->stream>>>(
            J, Fz, 1.0 / lambda, z_lo, z_hi, (const double2*)c, (const double2*)gamma, dir, z, (double2*)W);
}

// ------------------------------------------------------------------------------------------
// a-3 twiddles: Ft[f*N + i] = exp(i k s_f x_i) = exp(i 2 pi (f - nfreq/2) x_i / X)   (eq. 6, eq. 10)
template <typename T>
__global__ void k_twiddles(int nfreq, int64_t N, const double* __restrict__ coord, double inv_period,
                           typename C2<T>::type* __restrict__ Ft)
{
    using T2 = typename C2<T>::type;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)nfreq * N) return;
    const int64_t f = idx / N, i = idx - f * N;
    double t = (double)(f - nfreq / 2) * (coord[i] * inv_period);
    t -= rint(t);
    double s, co;
    sincospi(2.0 * t, &s, &co);
    Ft[idx] = mk2<T2, T>((T)co, (T)s);
}

void launch_twiddles(scw_ctx* ctx, int dtype, int nfreq, int64_t N, const double* coord, double period,
                     void* Ft)
{
    const int64_t n = (int64_t)nfreq * N;
    const int threads = 256;
    const unsigned blocks = (unsigned)((n + threads - 1) / threads);
    KernelScope ks(ctx, KC_TWIDDLES);
    if (dtype == SCW_C64)
        k_twiddles<float><<<blocks, threads, 0, ctx->stream>>>(nfreq, N, coord, 1.0 / period, (float2*)Ft);
    else
        k_twiddles<double><<<blocks, threads, 0, ctx->stream>>>(nfreq, N, coord, 1.0 / period, (double2*)Ft);
}

// ------------------------------------------------------------------------------------------
// a-2 spectral assembly, CUDA-core version: one thread per row of V, TN z-columns in registers,
// W tiles broadcast from shared memory, optional split over the mode index with a reduce pass.
constexpr int ASM_THREADS = 128;
constexpr int ASM_KB = 32;

template <typename T, int TN>
__global__ void __launch_bounds__(ASM_THREADS)
k_simt_assemble(int64_t R, int64_t J, int64_t Fz, const typename C2<T>::type* __restrict__ V, int64_t ldV,
                const typename C2<T>::type* __restrict__ W, typename C2<T>::type* __restrict__ out,
                int64_t ld_out, int64_t split_stride, int64_t kchunk)
{
    using T2 = typename C2<T>::type;
    __shared__ T2 Ws[ASM_KB][TN];
    const int tid = threadIdx.x;
    const int64_t row = (int64_t)blockIdx.x * ASM_THREADS + tid;
    const int64_t n0 = (int64_t)blockIdx.y * TN;
    const int64_t j0 = (int64_t)blockIdx.z * kchunk;
    const int64_t j1 = min(J, j0 + kchunk);
    const bool active = row < R;
    const T2* __restrict__ Vrow = V + (active ? row : 0);

    T2 acc[TN];
#pragma unroll
    for (int n = 0; n < TN; ++n) acc[n] = mk2<T2, T>((T)0, (T)0);

    for (int64_t jb = j0; jb < j1; jb += ASM_KB) {
        __syncthreads();
        for (int idx = tid; idx < ASM_KB * TN; idx += ASM_THREADS) {
            const int jj = idx / TN, nn = idx - jj * TN;
            T2 w = mk2<T2, T>((T)0, (T)0);
            if (jb + jj < j1 && n0 + nn < Fz) w = W[(jb + jj) * Fz + n0 + nn];
            Ws[jj][nn] = w;
        }
        __syncthreads();
        const int jn = (int)min((int64_t)ASM_KB, j1 - jb);
        if (active) {
#pragma unroll 4
            for (int jj = 0; jj < jn; ++jj) {
                const T2 v = Vrow[(jb + jj) * ldV];
#pragma unroll
                for (int n = 0; n < TN; ++n) cfma(acc[n], v, Ws[jj][n]);
            }
        }
    }
    if (active) {
        T2* o = out + (int64_t)blockIdx.z * split_stride + row;
#pragma unroll
        for (int n = 0; n < TN; ++n)
            if (n0 + n < Fz) o[(n0 + n) * ld_out] = acc[n];
    }
}

template <typename T>
__global__ void k_reduce_splits(int64_t R, int64_t Fz, int nsplit, const typename C2<T>::type* __restrict__ part,
                                typename C2<T>::type* __restrict__ P, int64_t ldP)
{
    using T2 = typename C2<T>::type;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= R * Fz) return;
    const int64_t i = idx / R, r = idx - i * R;
    T2 s = mk2<T2, T>((T)0, (T)0);
    for (int k = 0; k < nsplit; ++k) {
        const T2 v = part[(int64_t)k * R * Fz + idx];
        s.x += v.x;
        s.y += v.y;
    }
    P[r + i * ldP] = s;
}

static int simt_assemble_tn(int dtype, int64_t Fz) { return dtype == SCW_C64 ? (Fz <= 16 ? 16 : 32) : (Fz <= 8 ? 8 : 16); }

static int simt_assemble_splits(int dtype, int64_t R, int64_t J, int64_t Fz, int sm_count)
{
    const int tn = simt_assemble_tn(dtype, Fz);
    const int64_t tiles = ((R + ASM_THREADS - 1) / ASM_THREADS) * ((Fz + tn - 1) / tn);
    int64_t want = (6LL * sm_count + tiles - 1) / tiles;
    const int64_t max_split = (J + 4 * ASM_KB - 1) / (4 * ASM_KB);
    if (want > max_split) want = max_split;
    if (want < 1) want = 1;
    if (want > 65535) want = 65535;
    return (int)want;
}

size_t simt_assemble_scratch(int dtype, int64_t R, int64_t J, int64_t Fz, int sm_count)
{
    const int ns = simt_assemble_splits(dtype, R, J, Fz, sm_count);
    const size_t es = dtype == SCW_C64 ? 8 : 16;
    return ns > 1 ? align_up((size_t)ns * R * Fz * es) : 0;
}

template <typename T, int TN>
static void run_simt_assemble(scw_ctx* ctx, int64_t R, int64_t J, int64_t Fz, const void* V, int64_t ldV,
                              const void* W, void* P, int64_t ldP, void* scratch, int ns)
{
    using T2 = typename C2<T>::type;
    int64_t kchunk = (J + ns - 1) / ns;
    kchunk = (kchunk + ASM_KB - 1) / ASM_KB * ASM_KB;
    ns = (int)((J + kchunk - 1) / kchunk);
    dim3 grid((unsigned)((R + ASM_THREADS - 1) / ASM_THREADS), (unsigned)((Fz + TN - 1) / TN), (unsigned)ns);
    if (ns == 1) {
        KernelScope ks(ctx, KC_ASSEMBLE);
        k_simt_assemble<T, TN><<<grid, ASM_THREADS, 0, ctx->stream>>>(R, J, Fz, (const T2*)V, ldV, (const T2*)W,
                                                                      (T2*)P, ldP, 0, kchunk);
    } else {
        {
            KernelScope ks(ctx, KC_ASSEMBLE);
            k_simt_assemble<T, TN><<<grid, ASM_THREADS, 0, ctx->stream>>>(R, J, Fz, (const T2*)V, ldV, (const T2*)W,
                                                                          (T2*)scratch, R, R * Fz, kchunk);
        }
        const int64_t n = R * Fz;
        KernelScope ks(ctx, KC_REDUCE);
        k_reduce_splits<T><<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(R, Fz, ns, (const T2*)scratch,
                                                                                 (T2*)P, ldP);
    }
}

void launch_simt_assemble(scw_ctx* ctx, int dtype, int64_t R, int64_t J, int64_t Fz, const void* V,
                          int64_t ldV, const void* W, void* P, int64_t ldP, void* scratch)
{
    const int ns = simt_assemble_splits(dtype, R, J, Fz, ctx->sm_count);
    const int tn = simt_assemble_tn(dtype, Fz);
    if (dtype == SCW_C64) {
        if (tn == 16) run_simt_assemble<float, 16>(ctx, R, J, Fz, V, ldV, W, P, ldP, scratch, ns);
        else run_simt_assemble<float, 32>(ctx, R, J, Fz, V, ldV, W, P, ldP, scratch, ns);
    } else {
        if (tn == 8) run_simt_assemble<double, 8>(ctx, R, J, Fz, V, ldV, W, P, ldP, scratch, ns);
        else run_simt_assemble<double, 16>(ctx, R, J, Fz, V, ldV, W, P, ldP, scratch, ns);
    }
}

// ------------------------------------------------------------------------------------------
// a-4 separable synthesis, CUDA-core version (eq. 10 factored over the rectangular (u,v) grid):
//   pass A  T[plane][u][k] = sum_v P_comp[u,v] Fy[k,v]       (plane = n*3 + comp)
//   pass B  E[plane][k][i] = sum_u Fx[i,u] T[plane][u][k]
constexpr int SYN_THREADS = 128;

template <typename T, int TU>
__global__ void __launch_bounds__(SYN_THREADS)
k_simt_synth_a(int U, int Vn, const typename C2<T>::type* __restrict__ P, int64_t ldP, int64_t Ny,
               const typename C2<T>::type* __restrict__ FyT, typename C2<T>::type* __restrict__ Tb)
{
    using T2 = typename C2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T2* Ps = reinterpret_cast<T2*>(smem_raw);               // [Vn][TU]
    const int tid = threadIdx.x;
    const int64_t plane = blockIdx.x;
    const int64_t n = plane / 3;
    const int comp = (int)(plane - n * 3);
    const int64_t k = (int64_t)blockIdx.y * SYN_THREADS + tid;
    const int u0 = blockIdx.z * TU;
    const int64_t M = (int64_t)U * Vn;
    const T2* __restrict__ Pc = P + n * ldP + comp * M;
    for (int idx = tid; idx < Vn * TU; idx += SYN_THREADS) {
        const int v = idx / TU, uu = idx - v * TU;
        Ps[idx] = (u0 + uu < U) ? Pc[(int64_t)v * U + u0 + uu] : mk2<T2, T>((T)0, (T)0);
    }
    __syncthreads();
    if (k >= Ny) return;
    T2 acc[TU];
#pragma unroll
    for (int uu = 0; uu < TU; ++uu) acc[uu] = mk2<T2, T>((T)0, (T)0);
#pragma unroll 2
    for (int v = 0; v < Vn; ++v) {
        const T2 f = FyT[(int64_t)v * Ny + k];
#pragma unroll
        for (int uu = 0; uu < TU; ++uu) cfma(acc[uu], f, Ps[v * TU + uu]);
    }
#pragma unroll
    for (int uu = 0; uu < TU; ++uu)
        if (u0 + uu < U) Tb[(plane * U + u0 + uu) * Ny + k] = acc[uu];
}

template <typename T, int TK>
__global__ void __launch_bounds__(SYN_THREADS)
k_simt_synth_b(int U, int64_t Nx, int64_t Ny, const typename C2<T>::type* __restrict__ FxT,
               const typename C2<T>::type* __restrict__ Tb, typename C2<T>::type* __restrict__ E,
               int64_t s_comp, int64_t s_z, int64_t s_y, int64_t s_x)
{
    using T2 = typename C2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T2* Ts = reinterpret_cast<T2*>(smem_raw);               // [U][TK]
    const int tid = threadIdx.x;
    const int64_t plane = blockIdx.x;
    const int64_t n = plane / 3;
    const int comp = (int)(plane - n * 3);
    const int64_t i = (int64_t)blockIdx.y * SYN_THREADS + tid;
    const int64_t k0 = (int64_t)blockIdx.z * TK;
    for (int idx = tid; idx < U * TK; idx += SYN_THREADS) {
        const int u = idx / TK, kk = idx - u * TK;
        Ts[idx] = (k0 + kk < Ny) ? Tb[(plane * U + u) * Ny + k0 + kk] : mk2<T2, T>((T)0, (T)0);
    }
    __syncthreads();
    if (i >= Nx) return;
    T2 acc[TK];
#pragma unroll
    for (int kk = 0; kk < TK; ++kk) acc[kk] = mk2<T2, T>((T)0, (T)0);
#pragma unroll 2
    for (int u = 0; u < U; ++u) {
        const T2 f = FxT[(int64_t)u * Nx + i];
#pragma unroll
        for (int kk = 0; kk < TK; ++kk) cfma(acc[kk], f, Ts[u * TK + kk]);
    }
    T2* o = E + comp * s_comp + n * s_z + i * s_x;
#pragma unroll
    for (int kk = 0; kk < TK; ++kk)
        if (k0 + kk < Ny) o[(k0 + kk) * s_y] = acc[kk];
}

size_t simt_synth_scratch(int dtype, int U, int64_t Fz, int64_t Ny)
{
    const size_t es = dtype == SCW_C64 ? 8 : 16;
    return align_up((size_t)Fz * 3 * U * Ny * es);
}

template <typename T>
static void run_simt_synth(scw_ctx* ctx, int U, int Vn, int64_t Fz, const void* P, int64_t ldP, int64_t Nx,
                           const void* FxT, int64_t Ny, const void* FyT, void* E, const int64_t s[4],
                           void* scratch)
{
    using T2 = typename C2<T>::type;
    constexpr int TU = 8, TK = 16;
    const int64_t planes = Fz * 3;
    // gridDim.x carries the plane index (up to 2^31-1)
    dim3 ga((unsigned)planes, (unsigned)((Ny + SYN_THREADS - 1) / SYN_THREADS), (unsigned)((U + TU - 1) / TU));
    {
        KernelScope ks(ctx, KC_SYNTH_A);
        k_simt_synth_a<T, TU><<<ga, SYN_THREADS, (size_t)Vn * TU * sizeof(T2), ctx->stream>>>(
            U, Vn, (const T2*)P, ldP, Ny, (const T2*)FyT, (T2*)scratch);
    }
    dim3 gb((unsigned)planes, (unsigned)((Nx + SYN_THREADS - 1) / SYN_THREADS), (unsigned)((Ny + TK - 1) / TK));
    KernelScope ks(ctx, KC_SYNTH_B);
    k_simt_synth_b<T, TK><<<gb, SYN_THREADS, (size_t)U * TK * sizeof(T2), ctx->stream>>>(
        U, Nx, Ny, (const T2*)FxT, (const T2*)scratch, (T2*)E, s[0], s[1], s[2], s[3]);
}

void launch_simt_synth(scw_ctx* ctx, int dtype, int U, int Vn, int64_t Fz, const void* P, int64_t ldP,
                       int64_t Nx, const void* FxT, int64_t Ny, const void* FyT, void* E,
                       const int64_t strides[4], void* scratch)
{
    if (dtype == SCW_C64) run_simt_synth<float>(ctx, U, Vn, Fz, P, ldP, Nx, FxT, Ny, FyT, E, strides, scratch);
    else run_simt_synth<double>(ctx, U, Vn, Fz, P, ldP, Nx, FxT, Ny, FyT, E, strides, scratch);
}

// ------------------------------------------------------------------------------------------
// NEXT-3 detector, general path: I[n][k][i] = sum_comp |E[n][comp][k][i]|^2 from a planar E (the tensor-core synthesis
// fuses this into its epilogue instead).
template <typename T>
__global__ void k_intensity(int64_t Fz, int64_t Ny, int64_t Nx, const typename C2<T>::type* __restrict__ E,
                            T* __restrict__ I, int64_t s_z, int64_t s_y, int64_t s_x)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t plane = Nx * Ny;
    if (idx >= Fz * plane) return;
    const int64_t n = idx / plane, rem = idx - n * plane;
    const int64_t k = rem / Nx, i = rem - k * Nx;
    T acc = 0;
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
        const typename C2<T>::type e = E[(n * 3 + comp) * plane + rem];
        acc += e.x * e.x + e.y * e.y;
    }
    I[n * s_z + k * s_y + i * s_x] = acc;
}

void launch_intensity(scw_ctx* ctx, int dtype, int64_t Fz, int64_t Ny, int64_t Nx, const void* E, void* I,
                      const int64_t s3[3])
{
    const int64_t n = Fz * Ny * Nx;
    KernelScope ks(ctx, KC_MISC);
    if (dtype == SCW_C64)
        k_intensity<float><<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(Fz, Ny, Nx, (const float2*)E, (float*)I,
                                                                                   s3[0], s3[1], s3[2]);
    else
        k_intensity<double><<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(Fz, Ny, Nx, (const double2*)E, (double*)I,
                                                                                    s3[0], s3[1], s3[2]);
}

// NEXT-3 detector, general path: window sum of the intensity on a plane, one block per z plane, fixed reduction tree.
template <typename T>
__global__ void __launch_bounds__(256) k_window_sum(int64_t Ny, int64_t Nx, const typename C2<T>::type* __restrict__ E,
                                                   int64_t x0, int64_t x1, int64_t y0, int64_t y1, T* __restrict__ S)
{
    __shared__ T red[256];
    const int64_t n = blockIdx.x, plane = Nx * Ny;
    const int64_t wx = x1 - x0, cnt = wx * (y1 - y0);
    T acc = 0;
    for (int64_t i = threadIdx.x; i < cnt; i += 256) {
        const int64_t k = y0 + i / wx, ix = x0 + i % wx;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            const typename C2<T>::type e = E[(n * 3 + comp) * plane + k * Nx + ix];
            acc += e.x * e.x + e.y * e.y;
        }
    }
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) S[n] = red[0];
}

void launch_window_sum(scw_ctx* ctx, int dtype, int64_t Fz, int64_t Ny, int64_t Nx, const void* E, const int64_t win[4], void* S)
{
    KernelScope ks(ctx, KC_MISC);
    if (dtype == SCW_C64)
        k_window_sum<float><<<(unsigned)Fz, 256, 0, ctx->stream>>>(Ny, Nx, (const float2*)E, win[0], win[1], win[2], win[3], (float*)S);
    else
        k_window_sum<double><<<(unsigned)Fz, 256, 0, ctx->stream>>>(Ny, Nx, (const double2*)E, win[0], win[1], win[2], win[3], (double*)S);
}

// Absorbance A = -log10(S / S0) per entry and, optionally, of the band: -log10(sum w S / sum w S0).
template <typename T>
__global__ void __launch_bounds__(256) k_absorbance(int64_t n, const T* __restrict__ S, const T* __restrict__ S0,
                                                   const T* __restrict__ w, T* __restrict__ A, T* __restrict__ band)
{
    __shared__ double rs[256], r0[256];
    double as = 0.0, a0 = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += 256) {
        const double s = (double)S[i], s0 = (double)S0[i], wi = w ? (double)w[i] : 1.0;
        if (A) A[i] = (T)(-log10(s / s0));
        as += wi * s;
        a0 += wi * s0;
    }
    rs[threadIdx.x] = as;
    r0[threadIdx.x] = a0;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { rs[threadIdx.x] += rs[threadIdx.x + o]; r0[threadIdx.x] += r0[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0 && band) band[0] = (T)(-log10(rs[0] / r0[0]));
}

void launch_absorbance(scw_ctx* ctx, int dtype, int64_t n, const void* S, const void* S0, const void* w, void* A, void* band)
{
    KernelScope ks(ctx, KC_MISC);
    if (dtype == SCW_C64)
        k_absorbance<float><<<1, 256, 0, ctx->stream>>>(n, (const float*)S, (const float*)S0, (const float*)w, (float*)A, (float*)band);
    else
        k_absorbance<double><<<1, 256, 0, ctx->stream>>>(n, (const double*)S, (const double*)S0, (const double*)w, (double*)A, (double*)band);
}

}  // namespace scw
