// V builder: from the eigenvector matrix Q of a layer's property matrix D (rows P_x, P_y, B_x, B_y in
// blocks of M, eq. 19-23) to the matrix V = T Q [diag(alpha)] the field evaluation consumes
// (PAPER.md:428-432): the P_x, P_y rows are copied and the P_z rows follow from eq. 33,
//
//     [P_z]_m = + sum_{m'} psi_{m'} { [s_y]_{m-m'} [b_x]_{m-m'} - [s_x]_{m-m'} [b_y]_{m-m'} }
//
// i.e.  P_z = Psi_c . G,  G = diag(s_y) Q_Bx - diag(s_x) Q_By,  Psi_c[m, m''] = psi_{m (-) m''}: the 2-D circular
// convolution with the Fourier coefficients of 1/n^2 written as an M x M by M x J complex GEMM (the paper's O(M^3 L)
// precompute).  Readings: c-19 the sign is + (the printed minus contradicts eq. 14), c-20 "m - m'" is the
// difference of the frequency vectors wrapped per axis onto the grid of eq. 6 (block-circulant Psi, eq. 21), c-21
// psi_m are Fourier-SERIES coefficients, 1/n^2(r) = sum_m psi_m exp(ik s_m . r).
// Three launches: circulant + prepared operand (one kernel each), then the GEMM on the tensor cores -- complex64 on the
// tcgen05 assembly kernel in its generic-GEMM mode (BF16x3), complex128 on the DMMA kernel, CUDA cores otherwise.
#include "scw_internal.h"

namespace scw {

template <typename T2> struct VbReal;
template <> struct VbReal<float2> { using type = float; };
template <> struct VbReal<double2> { using type = double; };

// Psi_c[m + m''*M] = psi[m (-) m''], column-major M x M
template <typename T2>
__global__ void k_vb_circulant(int U, int Vn, const T2* __restrict__ psi, T2* __restrict__ Pc)
{
    const int M = U * Vn;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)M * M) return;
    const int m = (int)(idx % M), mm = (int)(idx / M);
    const int u = m % U - U / 2, v = m / U - Vn / 2, u2 = mm % U - U / 2, v2 = mm / U - Vn / 2;
    const int du = ((u - u2 + U / 2) % U + U) % U - U / 2;
    const int dv = ((v - v2 + Vn / 2) % Vn + Vn) % Vn - Vn / 2;
    Pc[idx] = psi[(dv + Vn / 2) * U + du + U / 2];
}

// G[k*J + n] = alpha_n (s_y[k] Q[2M + k, n] - s_x[k] Q[3M + k, n])   (row-major M x J, through a 32 x 32 tile transpose)
// and the copied rows V[r, n] = alpha_n Q[r, n], r < 2M.
template <typename T2>
__global__ void __launch_bounds__(256) k_vb_prepare(int U, int Vn, double lam_over_X, double lam_over_Y, int64_t J,
                                                   const T2* __restrict__ Q, int64_t ldQ, const T2* __restrict__ alpha,
                                                   T2* __restrict__ G, T2* __restrict__ V, int64_t ldV)
{
    using T = typename VbReal<T2>::type;
    __shared__ T2 tile[32][33];
    const int M = U * Vn;
    const int64_t k0 = (int64_t)blockIdx.x * 32, n0 = (int64_t)blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;              // 32 x 8 threads
    for (int i = ty; i < 32; i += 8) {                                   // read: k fastest (contiguous in Q)
        const int64_t k = k0 + tx, n = n0 + i;
        T2 g;
        g.x = 0;
        g.y = 0;
        if (k < M && n < J) {
            const int u = (int)(k % U) - U / 2, v = (int)(k / U) - Vn / 2;
            const T sx = (T)(lam_over_X * u), sy = (T)(lam_over_Y * v);
            const T2 bx = Q[2 * (int64_t)M + k + n * ldQ], by = Q[3 * (int64_t)M + k + n * ldQ];
            T2 a;
            a.x = 1;
            a.y = 0;
            if (alpha) a = alpha[n];
            const T gr = sy * bx.x - sx * by.x, gi = sy * bx.y - sx * by.y;
            g.x = a.x * gr - a.y * gi;
            g.y = a.x * gi + a.y * gr;
            // the two copied rows of this (k, n): P_x and P_y
#pragma unroll
            for (int blk = 0; blk < 2; ++blk) {
                const T2 q = Q[(int64_t)blk * M + k + n * ldQ];
                T2 o;
                o.x = a.x * q.x - a.y * q.y;
                o.y = a.x * q.y + a.y * q.x;
                V[(int64_t)blk * M + k + n * ldV] = o;
            }
        }
        tile[i][tx] = g;
    }
    __syncthreads();
    for (int i = ty; i < 32; i += 8) {                                   // write: n fastest (contiguous in G)
        const int64_t k = k0 + i, n = n0 + tx;
        if (k < M && n < J) G[k * J + n] = tile[tx][i];
    }
}

static bool vb_use_tc(const scw_ctx* ctx, const scw_vbuild* vb, const void* Pc)
{
    const int64_t M = (int64_t)vb->U * vb->Vn;
    return ctx->path != SCW_PATH_SIMT && tc_assemble_supported(vb->dtype, M, M, vb->J, Pc, M) && 2 * M >= 128 && M >= 64;
}

size_t vbuild_scratch(const scw_ctx* ctx, const scw_vbuild* vb)
{
    const int64_t M = (int64_t)vb->U * vb->Vn;
    const size_t es = vb->dtype == SCW_C64 ? 8 : 16;
    size_t gemm;
    if (vb->dtype == SCW_C64 && ctx->path != SCW_PATH_SIMT && 2 * M >= 128 && M >= 64)
        gemm = tc_assemble_scratch(ctx, M, M, vb->J, 1);
    else if (ctx->path != SCW_PATH_SIMT && dmma_supported(vb->dtype))
        gemm = dmma_assemble_scratch(M, M, vb->J, ctx->sm_count);
    else
        gemm = simt_assemble_scratch(vb->dtype, M, M, vb->J, ctx->sm_count);
    return align_up((size_t)M * M * es) + align_up((size_t)M * vb->J * es) + align_up(gemm);
}

void launch_vbuild(scw_ctx* ctx, const scw_vbuild* vb, void* V, int64_t ldV, void* scratch)
{
    const int64_t M = (int64_t)vb->U * vb->Vn, J = vb->J;
    const size_t es = vb->dtype == SCW_C64 ? 8 : 16;
    Carver cv(scratch);
    void* Pc = cv.take((size_t)M * M * es);
    void* G = cv.take((size_t)M * J * es);
    {
        KernelScope ks(ctx, KC_VBUILD_PREP);
        const unsigned blocks = (unsigned)((M * M + 255) / 256);
        if (vb->dtype == SCW_C64) k_vb_circulant<float2><<<blocks, 256, 0, ctx->stream>>>(vb->U, vb->Vn, (const float2*)vb->psi, (float2*)Pc);
        else k_vb_circulant<double2><<<blocks, 256, 0, ctx->stream>>>(vb->U, vb->Vn, (const double2*)vb->psi, (double2*)Pc);
    }
    {
        KernelScope ks(ctx, KC_VBUILD_PREP);
        const dim3 grid((unsigned)((M + 31) / 32), (unsigned)((J + 31) / 32));
        if (vb->dtype == SCW_C64)
            k_vb_prepare<float2><<<grid, 256, 0, ctx->stream>>>(vb->U, vb->Vn, vb->lambda / vb->X, vb->lambda / vb->Y, J,
                                                                (const float2*)vb->Q, vb->ldQ, (const float2*)vb->alpha,
                                                                (float2*)G, (float2*)V, ldV);
        else
            k_vb_prepare<double2><<<grid, 256, 0, ctx->stream>>>(vb->U, vb->Vn, vb->lambda / vb->X, vb->lambda / vb->Y, J,
                                                                 (const double2*)vb->Q, vb->ldQ, (const double2*)vb->alpha,
                                                                 (double2*)G, (double2*)V, ldV);
    }
    // P_z rows: C [M x J] = Psi_c [M x M] . G [M x J], written into rows 2M .. 3M-1 of V
    void* C = static_cast<char*>(V) + (size_t)2 * M * es;
    if (vb_use_tc(ctx, vb, Pc)) {
        void* gs = cv.take(tc_assemble_scratch(ctx, M, M, J, 1));
        launch_tc_gemm(ctx, M, M, J, Pc, M, G, C, ldV, gs);
    } else if (ctx->path != SCW_PATH_SIMT && dmma_supported(vb->dtype)) {
        void* gs = cv.take(dmma_assemble_scratch(M, M, J, ctx->sm_count));
        launch_dmma_assemble(ctx, M, M, J, Pc, M, G, C, ldV, gs);
    } else {
        void* gs = cv.take(simt_assemble_scratch(vb->dtype, M, M, J, ctx->sm_count));
        launch_simt_assemble(ctx, vb->dtype, M, M, J, Pc, M, G, C, ldV, gs);
    }
}

}  // namespace scw
