// alpha propagation across the layers of a stack: eq. 24-26, PAPER.md:252-296,
//
//     alpha^(1) = Q'_1^-1 r_0,      alpha^(l) = Q'_l^-1 Q`_{l-1} alpha^(l-1),      r_L = Q`_L alpha^(L)
//     Q'_l = Qcheck^(l) + Qhat^(l) G(Gamma^(l), z_l, z_{l-1}) = Q^(l) diag(d'),   Q`_l = Qcheck G(Gamma, z_{l-1}, z_l) + Qhat = Q^(l) diag(d`)
//
// (symbols de-garbled per DESIGN.md reading c-7; Qcheck / Qhat = "+" / "-" columns).  Because G is diagonal, one layer is:
// solve Q^(l) y = r_{l-1} (dense complex LU of a 4M x 4M matrix), alpha = y / d', r_l = Q^(l) (d` o alpha).
// Everything runs in fp64 (complex64 inputs are widened; a 4356 x 4356 LU in fp32 would lose the 2e-4 bar):
//   LU      blocked right-looking with partial pivoting, panels of 64 columns:
//             k_lu_panel   one cooperative launch per panel; the panel's rows are spread over the CTAs (in shared memory),
//                          per column: local |.|_1 maximum, candidate row and diagonal row published -> ONE grid
//                          barrier -> pivot chosen, rows interchanged, scale + rank-1 update
//             k_lu_laswp   the panel's row interchanges applied to the columns outside the panel
//             k_lu_trsm    U12 = L11^-1 A12, one warp per column (also written row-major for the GEMM)
//             k_dmma_cgemm A22 -= L21 U12 on the FP64 tensor cores (scw_dmma.cu, 3M complex product)
//   solve   row interchanges, then blocked forward / backward substitution (k_trsv_block + k_trsv_update)
#include <algorithm>

#include "scw_internal.h"

namespace scw {

constexpr int LU_NB = 64;                  // panel width
constexpr int LU_RPC = 128;                // max panel rows per CTA (shared memory: 128 x 64 x 16 B = 128 KB)
constexpr int LU_THREADS = 256;
#ifndef LU_ROWS_WANTED
#define LU_ROWS_WANTED 32                   // panel rows per CTA aimed at (32, 64, 96, 128 measured: 32 is the fastest)
#endif

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cdiv(double2 a, double2 b)
{
    const double d = b.x * b.x + b.y * b.y;
    return make_double2((a.x * b.x + a.y * b.y) / d, (a.y * b.x - a.x * b.y) / d);
}
__device__ __forceinline__ unsigned lu_ld_acquire(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

struct LuPanel {
    double2* A;            // [ld x n] column-major, factored in place
    int64_t n, ld, k0;
    int nb, rpc;           // panel columns, rows per CTA
    int* piv;              // [n] pivot row of every column (global row index)
    unsigned* bar;         // grid barrier counter (zero at launch)
    double* slot_val;      // [2][grid] local maxima
    int* slot_row;         // [2][grid]
    double2* rowbuf;       // [2][grid + 1][LU_NB]: every CTA's candidate row, then the diagonal row (double-buffered by column parity)
    int* info;             // set to column + 1 on an exactly zero pivot (first one wins)
};

// Grid-wide barrier of a cooperative launch (all CTAs resident): monotone counter, the target advances by gridDim.x.
__device__ __forceinline__ void lu_grid_sync(unsigned* bar, unsigned& target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        unsigned spins = 0;
        while (lu_ld_acquire(bar) < target)
            if (++spins > (1u << 26)) __trap();                    // a protocol error reports a CUDA error instead of hanging
        __threadfence();
    }
    __syncthreads();
    target += gridDim.x;
}

__global__ void __launch_bounds__(LU_THREADS, 1) k_lu_panel(const LuPanel p)
{
    extern __shared__ __align__(16) unsigned char lu_smem[];
    double2* a = reinterpret_cast<double2*>(lu_smem);             // [nb][rpc] column-major block of this CTA's rows
    __shared__ double2 pr[LU_NB];                                 // pivot row of the current column
    __shared__ double red_v[LU_THREADS / 32];
    __shared__ int red_r[LU_THREADS / 32];
    __shared__ int s_piv, s_win;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nb = p.nb, rpc = p.rpc;
    const int64_t row0 = p.k0 + (int64_t)blockIdx.x * rpc;        // first global row of this CTA
    const int rows = (int)max((int64_t)0, min((int64_t)rpc, p.n - row0));
    unsigned target = gridDim.x;

    for (int idx = tid; idx < rows * nb; idx += LU_THREADS) {     // load: rows contiguous in memory
        const int r = idx % rows, c = idx / rows;
        a[c * rpc + r] = p.A[(p.k0 + c) * p.ld + row0 + r];
    }
    __syncthreads();

    for (int j = 0; j < nb; ++j) {
        const int par = j & 1;
        const int64_t gj = p.k0 + j;                              // global row / column of the diagonal
        // ---- 1. local maximum of |re| + |im| over this CTA's rows >= gj (ties: the smaller row); the candidate row itself
        // (all nb entries) is published with it, and the owner of the diagonal row publishes that row: ONE grid barrier per
        // column instead of two
        double bv = -1.0;
        int br = 0x7fffffff;
        for (int r = tid; r < rows; r += LU_THREADS) {
            if (row0 + r >= gj) {
                const double2 v = a[j * rpc + r];
                const double m = fabs(v.x) + fabs(v.y);
                if (m > bv) { bv = m; br = (int)(row0 + r); }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
            const int orow = __shfl_xor_sync(0xffffffffu, br, o);
            if (ov > bv || (ov == bv && orow < br)) { bv = ov; br = orow; }
        }
        if (lane == 0) { red_v[warp] = bv; red_r[warp] = br; }
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < LU_THREADS / 32; ++w)
                if (red_v[w] > bv || (red_v[w] == bv && red_r[w] < br)) { bv = red_v[w]; br = red_r[w]; }
            p.slot_val[par * gridDim.x + blockIdx.x] = bv;
            p.slot_row[par * gridDim.x + blockIdx.x] = br;
            s_piv = br;                                            // local candidate (0x7fffffff: none)
        }
        __syncthreads();
        double2* rows_par = p.rowbuf + (size_t)par * (gridDim.x + 1) * LU_NB;
        {
            const int lb = s_piv;
            if (lb != 0x7fffffff)
                for (int c = tid; c < nb; c += LU_THREADS) rows_par[(size_t)blockIdx.x * LU_NB + c] = a[c * rpc + (lb - (int)row0)];
            if (gj >= row0 && gj < row0 + rows)
                for (int c = tid; c < nb; c += LU_THREADS) rows_par[(size_t)gridDim.x * LU_NB + c] = a[c * rpc + (int)(gj - row0)];
        }
        lu_grid_sync(p.bar, target);
        // ---- 2. global pivot = the best candidate; interchange with the diagonal row
        if (warp == 0) {
            double gv = -1.0;
            int gr = 0x7fffffff, gc = 0;
            for (int c = lane; c < (int)gridDim.x; c += 32) {
                const double v = __ldcg(&p.slot_val[par * gridDim.x + c]);       // written by other SMs: L2, not L1
                const int r = __ldcg(&p.slot_row[par * gridDim.x + c]);
                if (v > gv || (v == gv && r < gr)) { gv = v; gr = r; gc = c; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double ov = __shfl_xor_sync(0xffffffffu, gv, o);
                const int orow = __shfl_xor_sync(0xffffffffu, gr, o);
                const int oc = __shfl_xor_sync(0xffffffffu, gc, o);
                if (ov > gv || (ov == gv && orow < gr)) { gv = ov; gr = orow; gc = oc; }
            }
            if (lane == 0) {
                // no candidate at all: every entry at or below the diagonal is NaN (`m > bv` is false for NaN), the normal
                // state of the columns after an exactly zero pivot (0/0) or of a Q that holds NaN.  Keep the diagonal row
                // (published in slot gridDim.x) so that the NaNs simply propagate into alpha, as the header promises.
                if (gr == 0x7fffffff) { gr = (int)gj; gc = (int)gridDim.x; }
                s_piv = gr;
                s_win = gc;
                if (blockIdx.x == 0) {
                    p.piv[gj] = gr;
                    if (!(gv > 0.0)) atomicCAS(p.info, 0, (int)gj + 1);
                }
            }
        }
        __syncthreads();
        const int64_t pv = s_piv;
        for (int c = tid; c < nb; c += LU_THREADS) pr[c] = __ldcg(&rows_par[(size_t)s_win * LU_NB + c]);
        if (pv != gj) {
            if (pv >= row0 && pv < row0 + rows)
                for (int c = tid; c < nb; c += LU_THREADS) a[c * rpc + (int)(pv - row0)] = __ldcg(&rows_par[(size_t)gridDim.x * LU_NB + c]);
            if (gj >= row0 && gj < row0 + rows)
                for (int c = tid; c < nb; c += LU_THREADS) a[c * rpc + (int)(gj - row0)] = __ldcg(&rows_par[(size_t)s_win * LU_NB + c]);
        }
        __syncthreads();
        const double2 pivot = pr[j];
        const int r_first = (int)max((int64_t)0, gj + 1 - row0);  // rows strictly below the diagonal
        for (int r = r_first + tid; r < rows; r += LU_THREADS) a[j * rpc + r] = cdiv(a[j * rpc + r], pivot);
        __syncthreads();
        const int nr = rows - r_first;
        if (nr > 0) {
            for (int idx = tid; idx < nr * (nb - j - 1); idx += LU_THREADS) {
                const int r = r_first + idx % nr, c = j + 1 + idx / nr;
                const double2 l = a[j * rpc + r], u = pr[c];
                double2 v = a[c * rpc + r];
                v.x -= l.x * u.x - l.y * u.y;
                v.y -= l.x * u.y + l.y * u.x;
                a[c * rpc + r] = v;
            }
        }
        __syncthreads();
    }
    for (int idx = tid; idx < rows * nb; idx += LU_THREADS) {
        const int r = idx % rows, c = idx / rows;
        p.A[(p.k0 + c) * p.ld + row0 + r] = a[c * rpc + r];
    }
}

// Row interchanges of panel [k0, k0 + nb) applied, in order, to every column outside the panel.  A thread per column
// replaying the nb interchanges one after the other is a chain of nb dependent round trips to memory (47 us per panel at
// n = 4356).  Instead every block replays them once on an index array in shared memory (idx[r] = the row whose content ends
// up in row r), which leaves at most 2 nb rows to move (the diagonal rows and the pivot rows); thread = (move, half of the
// block's LSW_COLS columns) then loads its values -- all independent --, the block synchronises, and the values are stored:
// two round trips.  Shared memory: n ints.
constexpr int LSW_COLS = 32;                                       // columns per block
__global__ void __launch_bounds__(256) k_lu_laswp(double2* __restrict__ A, int64_t n, int64_t ld, int64_t k0, int nb,
                                                  const int* __restrict__ piv)
{
    extern __shared__ int lsw_idx[];
    const int tid = threadIdx.x;
    for (int64_t i = tid; i < n; i += 256) lsw_idx[i] = (int)i;
    __syncthreads();
    if (tid == 0)
        for (int j = 0; j < nb; ++j) {
            const int r = (int)k0 + j, q = piv[r];
            if (q != r && q >= 0 && q < n) { const int t = lsw_idx[r]; lsw_idx[r] = lsw_idx[q]; lsw_idx[q] = t; }
        }
    __syncthreads();
    const int m = tid & 127, half = tid >> 7;                      // LU_NB <= 64: at most 128 rows change
    int dst = -1;
    if (m < nb) dst = (int)k0 + m;
    else if (m < 2 * nb) {
        dst = piv[k0 + m - nb];
        if (dst < k0 + nb || dst >= n) dst = -1;                   // a pivot inside the diagonal block: covered by m < nb
    }
    const int src = dst >= 0 ? lsw_idx[dst] : -1;
    const bool active = dst >= 0 && src != dst;                    // (the same pivot row twice: two threads move the same value)
    constexpr int PER = LSW_COLS / 2;
    double2 v[PER];
    int64_t col[PER];
#pragma unroll
    for (int e = 0; e < PER; ++e) {
        int64_t c = (int64_t)blockIdx.x * LSW_COLS + half * PER + e;
        if (c >= k0) c += nb;                                      // skip the panel's own columns
        col[e] = c < n ? c : -1;
        if (active && col[e] >= 0) v[e] = A[col[e] * ld + src];
    }
    __syncthreads();                                               // every value of the block's columns is read before any is written
#pragma unroll
    for (int e = 0; e < PER; ++e)
        if (active && col[e] >= 0) A[col[e] * ld + dst] = v[e];
}

// U12 = L11^-1 A12 (L11 unit lower, nb x nb): one warp per column of A12, lane l holds rows l and l + 32.
// Also written row-major (Ut[k*ncols + c]) as the B operand of the trailing GEMM.
__global__ void __launch_bounds__(256) k_lu_trsm(double2* __restrict__ A, int64_t n, int64_t ld, int64_t k0, int nb,
                                                 double2* __restrict__ Ut)
{
    extern __shared__ __align__(16) unsigned char trsm_smem[];
    double2* L = reinterpret_cast<double2*>(trsm_smem);           // column-major nb x nb (64 KB: dynamic)
    for (int idx = threadIdx.x; idx < nb * nb; idx += 256) L[idx] = A[(k0 + idx / nb) * ld + k0 + idx % nb];
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int64_t ncols = n - k0 - nb;
    const int64_t c = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (c >= ncols) return;
    double2* col = A + (k0 + nb + c) * ld + k0;
    double2 x0 = lane < nb ? col[lane] : make_double2(0.0, 0.0);
    double2 x1 = lane + 32 < nb ? col[lane + 32] : make_double2(0.0, 0.0);
    for (int k = 0; k < nb; ++k) {
        const double2 src = k < 32 ? x0 : x1;
        const double2 xk = make_double2(__shfl_sync(0xffffffffu, src.x, k & 31), __shfl_sync(0xffffffffu, src.y, k & 31));
        if (lane > k && lane < nb) {
            const double2 l = L[k * nb + lane];
            x0.x -= l.x * xk.x - l.y * xk.y;
            x0.y -= l.x * xk.y + l.y * xk.x;
        }
        if (lane + 32 > k && lane + 32 < nb) {
            const double2 l = L[k * nb + lane + 32];
            x1.x -= l.x * xk.x - l.y * xk.y;
            x1.y -= l.x * xk.y + l.y * xk.x;
        }
    }
    if (lane < nb) { col[lane] = x0; Ut[(int64_t)lane * ncols + c] = x0; }
    if (lane + 32 < nb) { col[lane + 32] = x1; Ut[(int64_t)(lane + 32) * ncols + c] = x1; }
}

// ---- solves with the factored matrix ---------------------------------------------------------------------
// dst = P src for the row interchanges piv (applied in order): the interchanges are replayed on an index array in shared
// memory by one thread (n steps of shared-memory latency), then the vector is gathered in parallel.
__global__ void __launch_bounds__(256) k_lu_apply_piv(int64_t n, const int* __restrict__ piv, const double2* __restrict__ src,
                                                     double2* __restrict__ dst)
{
    extern __shared__ int lu_perm[];                               // [n] perm | [n] piv
    int* perm = lu_perm;
    int* pv = lu_perm + n;
    for (int64_t i = threadIdx.x; i < n; i += 256) { perm[i] = (int)i; pv[i] = piv[i]; }
    __syncthreads();
    if (threadIdx.x == 0)
        for (int64_t r = 0; r < n; ++r) {
            const int q = pv[r];
            if (q != r && q >= 0 && q < n) { const int t = perm[r]; perm[r] = perm[q]; perm[q] = t; }
        }
    __syncthreads();
    for (int64_t i = threadIdx.x; i < n; i += 256) dst[i] = src[perm[i]];
}

// Diagonal block [k0, k0 + nb) of the forward (unit lower) or backward (upper) substitution: the nb x nb block is staged in
// shared memory by the whole CTA (the substitution itself is a chain of nb dependent steps: it must not wait on global
// memory at every step), then one warp solves.
__global__ void __launch_bounds__(256) k_trsv_block(const double2* __restrict__ A, int64_t ld, int64_t k0, int nb, int upper,
                                                    double2* __restrict__ x)
{
    extern __shared__ __align__(16) unsigned char trsv_smem[];
    double2* T = reinterpret_cast<double2*>(trsv_smem);            // column-major nb x nb
    __shared__ double2 xs[LU_NB];
    for (int i0 = 0; i0 < nb * nb; i0 += 256 * 8) {     // eight independent loads per thread in flight
        double2 v[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int idx = i0 + e * 256 + threadIdx.x;
            if (idx < nb * nb) v[e] = A[(k0 + idx / nb) * ld + k0 + idx % nb];
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int idx = i0 + e * 256 + threadIdx.x;
            if (idx < nb * nb) T[idx] = v[e];
        }
    }
    for (int i = threadIdx.x; i < nb; i += 256) xs[i] = x[k0 + i];
    __syncthreads();
    if (threadIdx.x >= 32) return;
    const int lane = threadIdx.x;
    if (!upper) {
        for (int k = 0; k < nb; ++k) {
            const double2 xk = xs[k];
            for (int i = k + 1 + lane; i < nb; i += 32) {
                const double2 l = T[k * nb + i];
                xs[i].x -= l.x * xk.x - l.y * xk.y;
                xs[i].y -= l.x * xk.y + l.y * xk.x;
            }
            __syncwarp();
        }
    } else {
        for (int k = nb - 1; k >= 0; --k) {
            if (lane == 0) xs[k] = cdiv(xs[k], T[k * nb + k]);
            __syncwarp();
            const double2 xk = xs[k];
            for (int i = lane; i < k; i += 32) {
                const double2 u = T[k * nb + i];
                xs[i].x -= u.x * xk.x - u.y * xk.y;
                xs[i].y -= u.x * xk.y + u.y * xk.x;
            }
            __syncwarp();
        }
    }
    for (int i = lane; i < nb; i += 32) x[k0 + i] = xs[i];
}

// x[r] -= sum_{k in [k0, k0+nb)} A[r, k] x[k] for r in [r0, r1): one thread per row (rows are contiguous in memory).
__global__ void __launch_bounds__(256) k_trsv_update(const double2* __restrict__ A, int64_t ld, int64_t k0, int nb, int64_t r0,
                                                    int64_t r1, double2* __restrict__ x)
{
    __shared__ double2 xk[LU_NB];
    for (int i = threadIdx.x; i < nb; i += 256) xk[i] = x[k0 + i];
    __syncthreads();
    const int64_t r = r0 + (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (r >= r1) return;
    double2 acc = x[r];
    int k = 0;
    for (; k + 8 <= nb; k += 8) {                       // eight independent loads in flight (one per round trip otherwise)
        double2 a[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) a[e] = A[(k0 + k + e) * ld + r];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            acc.x -= a[e].x * xk[k + e].x - a[e].y * xk[k + e].y;
            acc.y -= a[e].x * xk[k + e].y + a[e].y * xk[k + e].x;
        }
    }
    for (; k < nb; ++k) {
        const double2 a = A[(k0 + k) * ld + r];
        acc.x -= a.x * xk[k].x - a.y * xk[k].y;
        acc.y -= a.x * xk[k].y + a.y * xk[k].x;
    }
    x[r] = acc;
}

// ---- layer bookkeeping -------------------------------------------------------------------------------------
template <typename T2>
__global__ void k_alpha_widen(int64_t n, int64_t ldQ, const T2* __restrict__ Q, double2* __restrict__ A)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * n) return;
    const int64_t r = idx % n, c = idx / n;
    const T2 v = Q[c * ldQ + r];
    A[idx] = make_double2((double)v.x, (double)v.y);
}

template <typename T2>
__global__ void k_alpha_vec_in(int64_t n, const T2* __restrict__ src, double2* __restrict__ dst)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = make_double2((double)src[i].x, (double)src[i].y);
}

// G(Gamma_j, z_from, z_to) = exp(i k (z_to - z_from) Gamma_j) (eq. 7), phase reduced in fp64
__device__ __forceinline__ double2 alpha_green(double2 g, double dz_over_lambda)
{
    double t = g.x * dz_over_lambda;
    t -= rint(t);
    double s, c;
    sincospi(2.0 * t, &s, &c);
    const double a = exp(-6.283185307179586476925 * g.y * dz_over_lambda);
    return make_double2(a * c, a * s);
}

// alpha_j = y_j / d'_j (written in the caller's dtype) and w_j = d`_j alpha_j (the operand of r_l = Q w)
template <typename T2>
__global__ void k_alpha_scale(int64_t n, double t_over_lambda, const double2* __restrict__ gamma, const int8_t* __restrict__ dir,
                              const double2* __restrict__ y, T2* __restrict__ alpha, double2* __restrict__ w)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double2 g = gamma[j];
    const bool plus = dir ? dir[j] > 0 : (g.y > 0.0 || (g.y == 0.0 && g.x >= 0.0));
    double2 a = y[j];
    double2 wj;
    if (plus) {                                   // d' = 1, d` = G(Gamma, z_{l-1}, z_l)
        wj = cmul(alpha_green(g, t_over_lambda), a);
    } else {                                      // d' = G(Gamma, z_l, z_{l-1}), d` = 1
        a = cdiv(a, alpha_green(g, -t_over_lambda));
        wj = a;
    }
    T2 o;
    o.x = a.x;
    o.y = a.y;
    alpha[j] = o;
    w[j] = wj;
}

// r = Q w with the caller's Q (either dtype), fp64 accumulation.  grid = (row blocks, MV_SLICES column slices): every CTA
// writes the partial sums of its slice, k_alpha_matvec_sum adds the slices in a fixed order (deterministic).
constexpr int MV_SLICES = 16;
template <typename T2>
__global__ void __launch_bounds__(256) k_alpha_matvec(int64_t n, int64_t ldQ, const T2* __restrict__ Q, const double2* __restrict__ w,
                                                     double2* __restrict__ part)
{
    __shared__ double2 ws[256];
    const int64_t row = (int64_t)blockIdx.x * 256 + threadIdx.x;
    const int64_t per = (n + MV_SLICES - 1) / MV_SLICES, c_begin = blockIdx.y * per, c_end = min(n, c_begin + per);
    double2 acc = make_double2(0.0, 0.0);
    for (int64_t c0 = c_begin; c0 < c_end; c0 += 256) {
        __syncthreads();
        if (c0 + threadIdx.x < c_end) ws[threadIdx.x] = w[c0 + threadIdx.x];
        __syncthreads();
        const int cn = (int)min((int64_t)256, c_end - c0);
        if (row < n)
            for (int c = 0; c < cn; ++c) {
                const T2 q = Q[(c0 + c) * ldQ + row];
                acc.x += (double)q.x * ws[c].x - (double)q.y * ws[c].y;
                acc.y += (double)q.x * ws[c].y + (double)q.y * ws[c].x;
            }
    }
    if (row < n) part[(int64_t)blockIdx.y * n + row] = acc;
}

__global__ void k_alpha_matvec_sum(int64_t n, const double2* __restrict__ part, double2* __restrict__ r)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double2 acc = make_double2(0.0, 0.0);
    for (int s = 0; s < MV_SLICES; ++s) {
        acc.x += part[(int64_t)s * n + i].x;
        acc.y += part[(int64_t)s * n + i].y;
    }
    r[i] = acc;
}

template <typename T2>
__global__ void k_alpha_vec_out(int64_t n, const double2* __restrict__ src, T2* __restrict__ dst)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    T2 o;
    o.x = src[i].x;
    o.y = src[i].y;
    dst[i] = o;
}

// ---- host side ------------------------------------------------------------------------------------------------
static int lu_grid(const scw_ctx* ctx, int64_t rows, int* rpc)
{
    int g = (int)((rows + LU_RPC - 1) / LU_RPC);
    const int want = (int)std::min<int64_t>(ctx->sm_count, (rows + LU_ROWS_WANTED - 1) / LU_ROWS_WANTED);
    if (g < want) g = want;
    if (g < 1) g = 1;
    *rpc = (int)((rows + g - 1) / g);
    return g;
}

// rows of a panel per CTA <= LU_RPC (shared memory) and the interchange replay holds 8 n bytes of shared memory
static size_t lu_misc_bytes(const scw_ctx* ctx)
{
    return 64 + align_up((size_t)2 * ctx->sm_count * 12, 64) + (size_t)2 * (ctx->sm_count + 1) * LU_NB * 16;
}

bool alpha_supported(const scw_ctx* ctx, int64_t n)
{
    return n >= 1 && (n + ctx->sm_count - 1) / ctx->sm_count <= LU_RPC && n * 8 <= 200 * 1024;
}

size_t alpha_scratch(const scw_ctx* ctx, int64_t n)
{
    return align_up((size_t)n * n * 16) + align_up((size_t)LU_NB * n * 16) + 3 * align_up((size_t)n * 16) + align_up((size_t)n * 4) +
           align_up(lu_misc_bytes(ctx));
}

void launch_propagate_alpha(scw_ctx* ctx, const scw_stack* st, const void* r0, void* const* alpha, void* rL, void* scratch)
{
    const int64_t n = st->n;
    const bool f32 = st->dtype == SCW_C64;
    Carver cv(scratch);
    double2* A = (double2*)cv.take((size_t)n * n * 16);
    double2* Ut = (double2*)cv.take((size_t)LU_NB * n * 16);
    double2* r = (double2*)cv.take((size_t)n * 16);
    double2* y = (double2*)cv.take((size_t)n * 16);
    double2* w = (double2*)cv.take((size_t)n * 16);
    int* piv = (int*)cv.take((size_t)n * 4);
    char* misc = (char*)cv.take(lu_misc_bytes(ctx));
    unsigned* bar = (unsigned*)misc;                       // [0]: barrier counter, [1]: info
    int* info = (int*)(misc + 4);
    double* slot_val = (double*)(misc + 64);               // [2][#SM]
    int* slot_row = (int*)(slot_val + 2 * ctx->sm_count);  // [2][#SM]
    double2* rowbuf = (double2*)(misc + 64 + align_up((size_t)2 * ctx->sm_count * 12, 64));   // [2][#SM + 1][LU_NB]
    const unsigned vb = (unsigned)((n + 255) / 256);
    {
        KernelScope ks(ctx, KC_ALPHA);
        if (f32) k_alpha_vec_in<float2><<<vb, 256, 0, ctx->stream>>>(n, (const float2*)r0, r);
        else k_alpha_vec_in<double2><<<vb, 256, 0, ctx->stream>>>(n, (const double2*)r0, r);
    }
    cudaFuncSetAttribute(k_lu_panel, cudaFuncAttributeMaxDynamicSharedMemorySize, LU_RPC * LU_NB * 16);
    cudaFuncSetAttribute(k_lu_trsm, cudaFuncAttributeMaxDynamicSharedMemorySize, LU_NB * LU_NB * 16);
    cudaFuncSetAttribute(k_trsv_block, cudaFuncAttributeMaxDynamicSharedMemorySize, LU_NB * LU_NB * 16);
    cudaFuncSetAttribute(k_lu_apply_piv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(n * 8));
    cudaFuncSetAttribute(k_lu_laswp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(n * 4));
    cudaMemsetAsync(misc, 0, 64, ctx->stream);
    for (int l = 0; l < st->n_layers; ++l) {
        const double t_over_lambda = (st->z_if[l + 1] - st->z_if[l]) / st->lambda;
        {
            KernelScope ks(ctx, KC_ALPHA);
            const unsigned nb2 = (unsigned)((n * n + 255) / 256);
            if (f32) k_alpha_widen<float2><<<nb2, 256, 0, ctx->stream>>>(n, st->ldQ, (const float2*)st->Q[l], A);
            else k_alpha_widen<double2><<<nb2, 256, 0, ctx->stream>>>(n, st->ldQ, (const double2*)st->Q[l], A);
        }
        // ---- LU of A (in place)
        for (int64_t k0 = 0; k0 < n; k0 += LU_NB) {
            const int nb = (int)std::min<int64_t>(LU_NB, n - k0);
            LuPanel p;
            p.A = A; p.n = n; p.ld = n; p.k0 = k0; p.nb = nb; p.piv = piv; p.bar = bar; p.slot_val = slot_val; p.slot_row = slot_row;
            p.rowbuf = rowbuf; p.info = info;
            const int grid = lu_grid(ctx, n - k0, &p.rpc);
            cudaMemsetAsync(bar, 0, 4, ctx->stream);
            {
                KernelScope ks(ctx, KC_ALPHA_PANEL);
                void* args[] = {&p};
                cudaLaunchCooperativeKernel((const void*)k_lu_panel, dim3(grid), dim3(LU_THREADS), args,
                                            (size_t)p.rpc * nb * 16, ctx->stream);
            }
            if (n > nb) {
                KernelScope ks(ctx, KC_ALPHA_LU);
                k_lu_laswp<<<(unsigned)((n - nb + LSW_COLS - 1) / LSW_COLS), 256, (size_t)n * 4, ctx->stream>>>(A, n, n, k0, nb, piv);
            }
            const int64_t rest = n - k0 - nb;
            if (rest > 0) {
                {
                    KernelScope ks(ctx, KC_ALPHA_LU);
                    k_lu_trsm<<<(unsigned)((rest + 7) / 8), 256, LU_NB * LU_NB * 16, ctx->stream>>>(A, n, n, k0, nb, Ut);
                }
                // A22 -= L21 U12
                launch_dmma_gemm_sub(ctx, rest, rest, nb, A + k0 * n + k0 + nb, n, Ut, rest, A + (k0 + nb) * n + k0 + nb, n);
            }
        }
        // ---- y = A^-1 r: interchanges, forward, backward
        {
            KernelScope ks(ctx, KC_ALPHA);
            k_lu_apply_piv<<<1, 256, (size_t)n * 8, ctx->stream>>>(n, piv, r, y);
        }
        for (int64_t k0 = 0; k0 < n; k0 += LU_NB) {
            const int nb = (int)std::min<int64_t>(LU_NB, n - k0);
            KernelScope ks(ctx, KC_ALPHA);
            k_trsv_block<<<1, 256, LU_NB * LU_NB * 16, ctx->stream>>>(A, n, k0, nb, 0, y);
            if (k0 + nb < n)
                k_trsv_update<<<(unsigned)((n - k0 - nb + 255) / 256), 256, 0, ctx->stream>>>(A, n, k0, nb, k0 + nb, n, y);
        }
        for (int64_t k0 = (n - 1) / LU_NB * LU_NB; k0 >= 0; k0 -= LU_NB) {
            const int nb = (int)std::min<int64_t>(LU_NB, n - k0);
            KernelScope ks(ctx, KC_ALPHA);
            k_trsv_block<<<1, 256, LU_NB * LU_NB * 16, ctx->stream>>>(A, n, k0, nb, 1, y);
            if (k0 > 0) k_trsv_update<<<(unsigned)((k0 + 255) / 256), 256, 0, ctx->stream>>>(A, n, k0, nb, 0, k0, y);
        }
        // ---- alpha = y / d', r = Q (d` o alpha)
        {
            KernelScope ks(ctx, KC_ALPHA);
            if (f32)
                k_alpha_scale<float2><<<vb, 256, 0, ctx->stream>>>(n, t_over_lambda, (const double2*)st->gamma[l], st->dir ? st->dir[l] : nullptr,
                                                                   y, (float2*)alpha[l], w);
            else
                k_alpha_scale<double2><<<vb, 256, 0, ctx->stream>>>(n, t_over_lambda, (const double2*)st->gamma[l], st->dir ? st->dir[l] : nullptr,
                                                                    y, (double2*)alpha[l], w);
        }
        {
            KernelScope ks(ctx, KC_ALPHA);
            const dim3 mv(vb, MV_SLICES);                  // the slice partials go to the U12 buffer (free outside the LU)
            if (f32) k_alpha_matvec<float2><<<mv, 256, 0, ctx->stream>>>(n, st->ldQ, (const float2*)st->Q[l], w, Ut);
            else k_alpha_matvec<double2><<<mv, 256, 0, ctx->stream>>>(n, st->ldQ, (const double2*)st->Q[l], w, Ut);
            k_alpha_matvec_sum<<<vb, 256, 0, ctx->stream>>>(n, Ut, r);
        }
    }
    if (rL) {
        KernelScope ks(ctx, KC_ALPHA);
        if (f32) k_alpha_vec_out<float2><<<vb, 256, 0, ctx->stream>>>(n, r, (float2*)rL);
        else k_alpha_vec_out<double2><<<vb, 256, 0, ctx->stream>>>(n, r, (double2*)rL);
    }
}

}  // namespace scw
