// complex128 contractions on the FP64 tensor cores (DMMA, mma.sync.m8n8k4.f64): spectral assembly P = V W (a-2,
// eq. 31 / PAPER.md:332-334, 428-432) and both passes of the separable synthesis E = F_x P F_y^T (a-4, eq. 10 /
// PAPER.md:119-124).  tcgen05 has no FP64 kind, so this path uses the warp-level mma.sync instruction.
//
// One batched complex GEMM kernel C[b] = A[b] B[b] serves the three uses.  The complex product runs as THREE real
// products ("3M"): T1 = A_r B_r, T2 = A_i B_i, T3 = (A_r + A_i)(B_r + B_i), C_r = T1 - T2, C_i = T3 - T1 - T2 --
// a quarter fewer tensor-core flops than the four-product form, which matters because this path is bound by the FP64
// tensor rate (37 TFLOP/s measured, equal to the FP64 FMA rate).  An 8x4 A fragment lane (g, t) loads the complex
// element A[m0 + g, k0 + t] with one 16-byte shared-memory load and forms (re, im, re + im); a 4x8 B fragment lane
// (t, g) does the same with B[k0 + t, n0 + g]; the row paddings below make both loads conflict-free.
// Every product and sum is fp64 (IEEE fma inside the tensor core).  3M is normwise as accurate as the direct product
// (error ~ a few ulp of |A||B| per term); the 1e-10 bar is relative to max|E|, five orders above that.
#include "scw_internal.h"

namespace scw {

constexpr int DG_TM = 64, DG_TN = 64;      // CTA tile in complex elements
constexpr int DG_KB = 16;                  // complex k per pipeline stage
constexpr int DG_STAGES = 3;
constexpr int DG_THREADS = 256;            // 8 warps = 4 (m) x 2 (n); warp tile 16 complex rows x 32 columns
constexpr int DG_LDA = DG_TM + 2;          // row strides (complex): 66 * 16 B = 32 B mod 128, so the four k rows of a
constexpr int DG_LDB = DG_TN + 2;          // fragment fall into disjoint banks
constexpr size_t DG_SMEM = (size_t)DG_STAGES * DG_KB * (DG_LDA + DG_LDB) * sizeof(double2);

struct DgParams {
    const double2* A; const double2* B; double2* C;
    int64_t M, N, K;
    int64_t sAk;                           // A(m,k) = A[k*sAk + m]         (m contiguous)
    int64_t sBk;                           // B(k,n) = B[k*sBk + n]         (n contiguous)
    int64_t sCm, sCn;                      // C(m,n) = C[m*sCm + n*sCn]
    int nb2;                               // batch b = b1*nb2 + b2
    int64_t bA1, bA2, bB1, bB2, bC1, bC2;  // batch strides (complex elements)
    int nsplit; int64_t kchunk;            // split k: split s covers [s*kchunk, min(K, (s+1)*kchunk)), C += s*splitC
    int64_t splitC;
    int sub;                               // 1: C -= A B (trailing update of the LU, scw_alpha.cu) instead of C = A B
};

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src, bool pred)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst_smem);
    const int sz = pred ? 16 : 0;          // src-size 0: the 16 bytes are zero-filled, src is not read
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(DG_THREADS, 2) k_dmma_cgemm(const DgParams p)
{
    extern __shared__ __align__(16) unsigned char dg_smem[];
    double2* As = reinterpret_cast<double2*>(dg_smem);                       // [stage][k][DG_LDA]
    double2* Bs = As + (size_t)DG_STAGES * DG_KB * DG_LDA;                   // [stage][k][DG_LDB]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, t = lane & 3;
    const int wm = warp & 3, wn = warp >> 2;
    const int64_t m0 = (int64_t)blockIdx.x * DG_TM, n0 = (int64_t)blockIdx.y * DG_TN;
    const int bz = blockIdx.z / p.nsplit, split = blockIdx.z - bz * p.nsplit;
    const int b1 = bz / p.nb2, b2 = bz - b1 * p.nb2;
    const double2* __restrict__ A = p.A + b1 * p.bA1 + b2 * p.bA2;
    const double2* __restrict__ B = p.B + b1 * p.bB1 + b2 * p.bB2;
    double2* __restrict__ C = p.C + b1 * p.bC1 + b2 * p.bC2 + split * p.splitC;
    const int64_t k_begin = (int64_t)split * p.kchunk;
    const int64_t k_end = min(p.K, k_begin + p.kchunk);
    const int nstages = (int)((k_end - k_begin + DG_KB - 1) / DG_KB);

    auto load_stage = [&](int s, int64_t k0) {
        double2* as = As + (size_t)s * DG_KB * DG_LDA;
        double2* bs = Bs + (size_t)s * DG_KB * DG_LDB;
#pragma unroll
        for (int i = 0; i < DG_KB * DG_TM / DG_THREADS; ++i) {
            const int id = tid + i * DG_THREADS, k = id / DG_TM, m = id - k * DG_TM;
            const bool ok = k0 + k < k_end && m0 + m < p.M;
            cp_async16(as + k * DG_LDA + m, ok ? A + (k0 + k) * p.sAk + m0 + m : A, ok);
        }
#pragma unroll
        for (int i = 0; i < DG_KB * DG_TN / DG_THREADS; ++i) {
            const int id = tid + i * DG_THREADS, k = id / DG_TN, n = id - k * DG_TN;
            const bool ok = k0 + k < k_end && n0 + n < p.N;
            cp_async16(bs + k * DG_LDB + n, ok ? B + (k0 + k) * p.sBk + n0 + n : B, ok);
        }
    };

    // accumulators of the three real products: [m tile][n tile][T1, T2, T3][2 columns]
    double acc[2][4][3][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < 3; ++q) acc[i][j][q][0] = acc[i][j][q][1] = 0.0;

    for (int s = 0; s < DG_STAGES - 1; ++s) {
        if (s < nstages) load_stage(s, k_begin + (int64_t)s * DG_KB);
        cp_async_commit();
    }
    // fragment addressing (complex elements): A lane (g,t): row g, k t; B lane (t,g): k t, column g
    const int a_off = t * DG_LDA + wm * 16 + g;
    const int b_off = t * DG_LDB + wn * 32 + g;

    for (int st = 0; st < nstages; ++st) {
        cp_async_wait<DG_STAGES - 2>();
        __syncthreads();
        {   // prefetch stage st + STAGES-1 into the slot freed by iteration st-1
            const int nx = st + DG_STAGES - 1;
            if (nx < nstages) load_stage(nx % DG_STAGES, k_begin + (int64_t)nx * DG_KB);
            cp_async_commit();
        }
        const double2* as = As + (size_t)(st % DG_STAGES) * DG_KB * DG_LDA + a_off;
        const double2* bs = Bs + (size_t)(st % DG_STAGES) * DG_KB * DG_LDB + b_off;
        auto k_step = [&](int k4) {                     // 4 complex k
            double2 a[2], b[4];
#pragma unroll
            for (int i = 0; i < 2; ++i) a[i] = as[k4 * 4 * DG_LDA + i * 8];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = bs[k4 * 4 * DG_LDB + j * 8];
            double asum[2], bsum[4];
#pragma unroll
            for (int i = 0; i < 2; ++i) asum[i] = a[i].x + a[i].y;
#pragma unroll
            for (int j = 0; j < 4; ++j) bsum[j] = b[j].x + b[j].y;
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    dmma884(acc[i][j][0][0], acc[i][j][0][1], a[i].x, b[j].x);
                    dmma884(acc[i][j][1][0], acc[i][j][1][1], a[i].y, b[j].y);
                    dmma884(acc[i][j][2][0], acc[i][j][2][1], asum[i], bsum[j]);
                }
        };
        const int64_t k_left = k_end - (k_begin + (int64_t)st * DG_KB);
        if (k_left >= DG_KB) {
#pragma unroll
            for (int k4 = 0; k4 < DG_KB / 4; ++k4) k_step(k4);
        } else {                                        // ragged last stage: only the k quads that hold data
            const int k4n = (int)((k_left + 3) / 4);
#pragma unroll 1
            for (int k4 = 0; k4 < k4n; ++k4) k_step(k4);
        }
    }
    cp_async_wait<0>();

    // C fragment: lane (g,t) holds rows m = .. + g, columns 2t and 2t+1 of T1, T2, T3
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int64_t m = m0 + wm * 16 + i * 8 + g;
        if (m >= p.M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int64_t n = n0 + wn * 32 + j * 8 + 2 * t + e;
                const double t1 = acc[i][j][0][e], t2 = acc[i][j][1][e], t3 = acc[i][j][2][e];
                if (n < p.N) {
                    double2* dst = C + m * p.sCm + n * p.sCn;
                    if (p.sub) {
                        const double2 old = *dst;
                        *dst = make_double2(old.x - (t1 - t2), old.y - (t3 - t1 - t2));
                    } else {
                        *dst = make_double2(t1 - t2, t3 - t1 - t2);
                    }
                }
            }
        }
    }
}

static void dg_launch(scw_ctx* ctx, int kc, const DgParams& p, int batch)
{
    cudaFuncSetAttribute(k_dmma_cgemm, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DG_SMEM);
    const dim3 grid((unsigned)((p.M + DG_TM - 1) / DG_TM), (unsigned)((p.N + DG_TN - 1) / DG_TN), (unsigned)(batch * p.nsplit));
    KernelScope ks(ctx, kc);
    k_dmma_cgemm<<<grid, DG_THREADS, DG_SMEM, ctx->stream>>>(p);
}

// ---- a-2 spectral assembly: P = V W, split over the mode index when the tile count cannot fill the GPU ----------
static int dg_assemble_splits(int64_t R, int64_t J, int64_t Fz, int sm_count)
{
    // the split count that fills whole waves of 2 resident CTAs per SM best (a 5 % over-subscription would
    // otherwise run a nearly empty second wave); more splits only cost partial-tile traffic
    const int64_t tiles = ((R + DG_TM - 1) / DG_TM) * ((Fz + DG_TN - 1) / DG_TN);
    const int64_t slots = 2LL * sm_count;
    int64_t max_split = (J + 8 * DG_KB - 1) / (8 * DG_KB);
    if (max_split > 64) max_split = 64;
    if (tiles >= 4 * slots || max_split <= 1) return 1;
    int best = 1;
    double best_eff = 0.0;
    for (int ns = 1; ns <= max_split; ++ns) {
        const int64_t ctas = tiles * ns, waves = (ctas + slots - 1) / slots;
        const double eff = (double)ctas / (double)(waves * slots) - 0.002 * ns;
        if (eff > best_eff) { best_eff = eff; best = ns; }
    }
    return best;
}

bool dmma_supported(int dtype) { return dtype == SCW_C128; }

// C [ldC x N] -= A [ldA x K] (column-major, M rows) . B [K x N] (row-major, ldB): the trailing update of the blocked LU.
void launch_dmma_gemm_sub(scw_ctx* ctx, int64_t M, int64_t N, int64_t K, const void* A, int64_t ldA, const void* B, int64_t ldB,
                          void* C, int64_t ldC)
{
    DgParams p = {};
    p.A = (const double2*)A;
    p.B = (const double2*)B;
    p.C = (double2*)C;
    p.M = M; p.N = N; p.K = K;
    p.sAk = ldA;
    p.sBk = ldB;
    p.sCm = 1; p.sCn = ldC;
    p.nb2 = 1;
    p.nsplit = 1;
    p.kchunk = (K + DG_KB - 1) / DG_KB * DG_KB;
    p.sub = 1;
    dg_launch(ctx, KC_ALPHA_LU, p, 1);
}

size_t dmma_assemble_scratch(int64_t R, int64_t J, int64_t Fz, int sm_count)
{
    const int ns = dg_assemble_splits(R, J, Fz, sm_count);
    return ns > 1 ? align_up((size_t)ns * R * Fz * sizeof(double2)) : 0;
}

__global__ void k_dmma_reduce_splits(int64_t R, int64_t Fz, int nsplit, const double2* __restrict__ part,
                                     double2* __restrict__ P, int64_t ldP)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= R * Fz) return;
    const int64_t i = idx / R, r = idx - i * R;
    double2 s = make_double2(0.0, 0.0);
    for (int k = 0; k < nsplit; ++k) {                                // fixed order: deterministic
        const double2 v = part[(int64_t)k * R * Fz + idx];
        s.x += v.x;
        s.y += v.y;
    }
    P[r + i * ldP] = s;
}

// W is the a-1 table W[j*Fz + i] (plane fastest) produced by launch_mode_weights.
void launch_dmma_assemble(scw_ctx* ctx, int64_t R, int64_t J, int64_t Fz, const void* V, int64_t ldV, const void* W,
                          void* P, int64_t ldP, void* scratch)
{
    int ns = dg_assemble_splits(R, J, Fz, ctx->sm_count);
    int64_t kchunk = (J + ns - 1) / ns;
    kchunk = (kchunk + DG_KB - 1) / DG_KB * DG_KB;
    ns = (int)((J + kchunk - 1) / kchunk);
    DgParams p = {};
    p.A = (const double2*)V;
    p.B = (const double2*)W;
    p.M = R; p.N = Fz; p.K = J;
    p.sAk = ldV;
    p.sBk = Fz;
    p.nb2 = 1;
    p.nsplit = ns;
    p.kchunk = kchunk;
    if (ns == 1) {
        p.C = (double2*)P; p.sCm = 1; p.sCn = ldP; p.splitC = 0;
        dg_launch(ctx, KC_ASSEMBLE_DMMA, p, 1);
        return;
    }
    p.C = (double2*)scratch; p.sCm = 1; p.sCn = R; p.splitC = R * Fz;
    dg_launch(ctx, KC_ASSEMBLE_DMMA, p, 1);
    const int64_t n = R * Fz;
    KernelScope ks(ctx, KC_REDUCE);
    k_dmma_reduce_splits<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(R, Fz, ns, (const double2*)scratch,
                                                                                (double2*)P, ldP);
}

// ---- a-4 separable synthesis: pass A  T[plane][u][k] = sum_v P_comp[u,v] Fy[k,v],  pass B  E[k][i] = sum_u Fx[i,u] T[u][k]
// FxT / FyT are the frequency-major a-3 tables of launch_twiddles; scratch holds T (simt_synth_scratch bytes).
void launch_dmma_synth(scw_ctx* ctx, int U, int Vn, int64_t Fz, const void* P, int64_t ldP, int64_t Nx, const void* FxT,
                       int64_t Ny, const void* FyT, void* E, const int64_t s[4], void* scratch)
{
    const int64_t M = (int64_t)U * Vn;
    // the planes go into gridDim.z (<= 65535): chunks of z
    const int64_t z_chunk = 65535 / 3;
    for (int64_t z0 = 0; z0 < Fz; z0 += z_chunk) {
        const int64_t nz = Fz - z0 < z_chunk ? Fz - z0 : z_chunk;
        double2* T = (double2*)scratch + z0 * 3 * U * Ny;
        DgParams a = {};
        a.A = (const double2*)P + z0 * ldP; a.sAk = U;                      // A(u, v) = P_comp[v*U + u]
        a.B = (const double2*)FyT; a.sBk = Ny;                              // B(v, k) = FyT[v*Ny + k]
        a.C = T; a.sCm = Ny; a.sCn = 1;                                     // C(u, k) = T[plane][u*Ny + k]
        a.M = U; a.N = Ny; a.K = Vn;
        a.nb2 = 3;
        a.bA1 = ldP; a.bA2 = M;
        a.bC1 = 3LL * U * Ny; a.bC2 = (int64_t)U * Ny;
        a.nsplit = 1; a.kchunk = (Vn + DG_KB - 1) / DG_KB * DG_KB;
        dg_launch(ctx, KC_SYNTH_A_DMMA, a, (int)(nz * 3));
        DgParams b = {};
        b.A = (const double2*)FxT; b.sAk = Nx;                              // A(i, u) = FxT[u*Nx + i]
        b.B = T; b.sBk = Ny;                                                // B(u, k) = T[plane][u*Ny + k]
        b.C = (double2*)E + z0 * s[1]; b.sCm = s[3]; b.sCn = s[2];          // C(i, k) = E[comp][z][k][i]
        b.M = Nx; b.N = Ny; b.K = U;
        b.nb2 = 3;
        b.bB1 = 3LL * U * Ny; b.bB2 = (int64_t)U * Ny;
        b.bC1 = s[1]; b.bC2 = s[0];
        b.nsplit = 1; b.kchunk = (U + DG_KB - 1) / DG_KB * DG_KB;
        dg_launch(ctx, KC_SYNTH_B_DMMA, b, (int)(nz * 3));
    }
}

}  // namespace scw
