// Separable Fourier synthesis E_comp(z) = F_x . P_comp(z) . F_y^T on the 5th-gen tensor cores, complex64.
//   E_comp(x_i, y_k, z_n) = sum_{u,v} P[comp*M + m(u,v), n] exp(i 2 pi (u x_i/X + v y_k/Y))     (eq. 10)
// exact because the spatial frequencies lie on a rectangular (u,v) grid (eq. 6).
//
// One persistent CTA owns a 128(x) x 128(y) output tile and walks the (z, comp) planes.  Per plane two chained
// real GEMMs run on tcgen05 with fp32 accumulators in TMEM, each as three bf16 products (hi*hi + hi*lo + lo*hi):
//   GEMM1  D1[y, 2u+c]        = sum_k A1[y, k] B1[2u+c, k]        A1 = (Fy_r, Fy_i) interleaved over k = 2v+c''
//                                                                  B1 = the plane's spectrum in "complex as real" form
//          -> D1 row y holds T[u, y] = sum_v P[u,v] Fy[y,v] as (Re, Im) pairs
//   GEMM2  D2[x, 2y+c]        = sum_k A2[x, k] B2[2y+c, k]        A2 = (Fx_r, Fx_i), B2 built from D1 in-kernel
// The frequencies are cut into chunks of at most 40 (K <= 80 per GEMM): GEMM1 accumulates the v chunks into D1,
// GEMM2 accumulates the u chunks into D2, so up to 80 x 80 frequencies run in one pass over the output.
// A1 (all v chunks) sits in shared memory; A2 (all u chunks) is written ONCE into TMEM and GEMM2 runs in TS mode
// (A from TMEM, B from shared memory), which halves the shared-memory operand traffic of the dominant GEMM.
// The 128 converter threads read their own D1 row from TMEM (tcgen05.ld), split it to bf16 hi/lo and write the two
// B2 rows (y,Re), (y,Im) of the K-major UMMA image; the 128 epilogue threads read D2 (lane = x) and store
// (Re, Im) pairs straight to E: a warp writes 256 contiguous bytes per y.  Twiddle and spectrum images are
// produced by two small pre-kernels and fetched with bulk async copies.
#include "scw_internal.h"
#include "scw_tc_common.cuh"
#include "scw_exterior.cuh"

namespace scw {

using namespace tc;

constexpr int TS_TILE = 128;               // output tile edge (x and y)
constexpr int TS_KMAX = 80;                // max padded K per chunk (= 2*chunk rounded up to 16)
constexpr int TS_FMAX = 80;                // max frequencies per axis (two chunks)
constexpr int TS_THREADS = 19 * 32;        // loader, GEMM2 issuer, 8 converter warps, 8 epilogue warps, GEMM1 issuer
constexpr int TS_GEMM1_WARP = 18;
constexpr int TS_TMEM_COLS = 512;
constexpr int TS_D2_COL = 0;               // D2[h] at columns h*128
constexpr int TS_D1_COL = 256;             // D1 at columns 256..256+N1, then A2 (per u chunk: hi K2p/2 | lo K2p/2 columns)
constexpr int TS_MAX_INST = 64;            // instances per grouped launch


struct TsWsumOut { float* S[TS_MAX_INST]; };

struct TsParams {
    const uint8_t* A1;     // [ty][vc][hi|lo] images of (Fy_r, Fy_i): 128 rows x K1p, K-major, LBO = 2048, SBO = 128
    const uint32_t* A2;    // [tx][uc][row][hi K2p/2 | lo K2p/2] packed bf16 pairs (cos, sin) of Fx: TMEM A-operand rows
    const uint8_t* B1;     // [plane][uc][vc][hi|lo] images: N1 rows x K1p, MN-major, LBO (k blocks) = N1*16, SBO (row blocks) = 128
    float2* E[TS_MAX_INST];   // output of every instance of the group
    int64_t s_comp, s_z, s_y, s_x;
    int64_t Nx, Ny;
    int planes;            // n_inst * Fz * 3 (global plane id = inst * planes_per_inst + n*3 + comp)
    int planes_per_inst;
    int K1p, K2p;          // padded 2*Vc, 2*Uc  (N1 == K2p)
    int nuc, nvc;          // frequency chunks along u and v
    int tiles_x, tiles_y, pair0, npairs;   // this launch covers tile pairs [pair0, pair0 + npairs)
    int* sched;            // [tile pair] next plane group to hand out (zeroed by the spectrum-image kernel)
    int group;             // planes per drawn unit: 1, or 3 (the components of one z) when the detector writes I
    // NEXT-3 detector (k_tc_synth<true>): no complex field is stored.
    int want_I;            // E[] point to float outputs I = sum_comp |E_comp|^2
    int acc_col;           // first of 128 TMEM columns holding the running sum over components, 0 = none (kept in the output)
    int d2_single;         // detector with 33..40 frequencies along u (one u chunk): D2 is ONE 128-column buffer shared by the two y halves
                           // (released as soon as it is in registers), its second half holds the running sum
    int b2_stages;         // 1, or 2 when shared memory holds two B2 buffers: the converters fill one while GEMM2 reads the other
    float* s_part;         // window sums: [plane][tile][16] partial sums of |E_comp|^2 over the window, NULL = not wanted
    int win_x0, win_x1, win_y0, win_y1;   // window (grid indices, half-open)
    unsigned long long* tl_slot;          // timeline ring slot of this launch (scw_profile_timeline), may be NULL
};

__host__ __device__ inline int ts_pad16(int v) { return (v + 15) / 16 * 16; }

// Chunking of one frequency axis: n chunks of `len` frequencies (the last may be shorter), padded K = Kp.
struct TsChunks { int n, len, Kp; };
__host__ __device__ inline TsChunks ts_chunks(int nfreq)
{
    TsChunks c;
    c.n = (2 * nfreq + TS_KMAX - 1) / TS_KMAX;
    c.len = (nfreq + c.n - 1) / c.n;
    c.Kp = ts_pad16(2 * c.len);
    return c;
}

// ---- pre-kernels ------------------------------------------------------------------------------------
// Twiddle operands (a-3) in one launch.  y axis: K-major UMMA images, for tile t, chunk ch, row r (coordinate index
// t*128 + r), k = 2f + c: c = 0 -> cos, c = 1 -> sin of 2 pi (ch*len + f - nfreq/2) coord / period; rows past N and
// frequencies past the axis are zero; hi image then lo image.  x axis: the same values as TMEM A-operand rows,
// row = [hi: Kp/2 words | lo: Kp/2 words], word f = bf16 pair (cos, sin).
struct TwAxis { int nfreq, nch, len, Kp, tiles; int64_t N; const double* coord; double inv_period; void* out; };

__global__ void k_tc_synth_twiddles(const TwAxis ay, const TwAxis ax, int blocks_y, int* __restrict__ zero, size_t n_zero)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_zero; i += (size_t)gridDim.x * blockDim.x)
        zero[i] = 0;                                                          // control block of the assembly that follows
    const bool is_y = (int)blockIdx.x < blocks_y;                            // one launch covers both axes
    const TwAxis& a = is_y ? ay : ax;
    const int64_t idx = (int64_t)(blockIdx.x - (is_y ? 0 : blocks_y)) * blockDim.x + threadIdx.x;   // (tile, chunk, r, f)
    const int kpairs = a.Kp / 2;
    if (idx >= (int64_t)a.tiles * a.nch * TS_TILE * kpairs) return;
    const int f = (int)(idx % kpairs);
    const int64_t tr = idx / kpairs;
    const int r = (int)(tr % TS_TILE);
    const int tc_ = (int)(tr / TS_TILE);                                      // tile * nch + chunk
    const int ch = tc_ % a.nch, t = tc_ / a.nch;
    const int64_t i = (int64_t)t * TS_TILE + r;
    const int fg = ch * a.len + f;
    float co = 0.f, si = 0.f;
    if (f < a.len && fg < a.nfreq && i < a.N) {
        double ph = (double)(fg - a.nfreq / 2) * (a.coord[i] * a.inv_period);  // turns, reduced in fp64; the bf16 hi/lo
        ph -= rint(ph);                                                         // split below keeps 2^-17: fp32 sincospi
        sincospif((float)(2.0 * ph), &si, &co);
    }
    uint32_t hi, lo;
    split_bf16x2(co, si, hi, lo);
    if (is_y) {
        const int k = 2 * f;
        const size_t img_bytes = (size_t)TS_TILE * a.Kp * 2;
        uint8_t* base = static_cast<uint8_t*>(a.out) + (size_t)tc_ * 2 * img_bytes;
        const size_t off = (size_t)(k >> 3) * 2048 + (size_t)(r >> 3) * 128 + (r & 7) * 16 + (k & 7) * 2;
        *reinterpret_cast<uint32_t*>(base + off) = hi;
        *reinterpret_cast<uint32_t*>(base + img_bytes + off) = lo;
    } else {
        uint32_t* row = static_cast<uint32_t*>(a.out) + ((size_t)tc_ * TS_TILE + r) * a.Kp;
        row[f] = hi;
        row[kpairs + f] = lo;
    }
}

// Spectrum images (GEMM1's B operand): image (plane, uc, vc), plane = n*3 + comp, row n' = 2ul + c, k = 2vl + c'' with
// u = uc*Uc + ul, v = vc*Vc + vl:   row (u,Re): (P_r, -P_i) over (k, k+1);  row (u,Im): (P_i, P_r)
// so that  D1[y, (u,c)] = sum_v Fy[y,v] P[u,v]  in real arithmetic.  The image is MN-MAJOR (no swizzle): element (n', k) at
//   (k/8)*(N1*16) + (n'/8)*128 + (k%8)*16 + (n'%8)*2      [core matrix = 8 k-rows of 16 bytes, 8 rows n' contiguous]
// so that consecutive u -- consecutive rows of P, which is what one thread block of the producer holds -- are contiguous
// in memory: the word at k = 2vl is the bf16 pair (P_r, P_i), the word at k + 1 (16 bytes on) is (-P_i, P_r).
__device__ __forceinline__ void ts_image_store(uint8_t* img_hi, size_t img_bytes, int N1, int ul, int vl, float pr, float pi)
{
    uint32_t H, L;
    split_bf16x2(pr, pi, H, L);
    const int k = 2 * vl, n = 2 * ul;
    uint8_t* dst = img_hi + (size_t)(k >> 3) * (N1 * 16) + (size_t)(n >> 3) * 128 + (k & 7) * 16 + (n & 7) * 2;
    *reinterpret_cast<uint32_t*>(dst) = H;
    *reinterpret_cast<uint32_t*>(dst + 16) = __byte_perm(H, 0, 0x1032) ^ 0x00008000u;       // (-P_i, P_r)
    *reinterpret_cast<uint32_t*>(dst + img_bytes) = L;
    *reinterpret_cast<uint32_t*>(dst + img_bytes + 16) = __byte_perm(L, 0, 0x1032) ^ 0x00008000u;
}

__global__ void k_tc_synth_pimage(int U, int Vn, int Uc, int Vc, int nuc, int nvc, int K1p, int N1, int planes,
                                  const float2* __restrict__ P, int64_t ldP, uint8_t* __restrict__ img,
                                  int* __restrict__ sched, int n_sched)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // (image, vl, ul), ul fastest
    for (int64_t i = idx; i < n_sched; i += (int64_t)gridDim.x * blockDim.x) sched[i] = 0;   // plane counters of the synthesis that follows
    const int half_n = N1 / 2, kpairs = K1p / 2;
    if (idx >= (int64_t)planes * nuc * nvc * half_n * kpairs) return;
    const int ul = (int)(idx % half_n);
    const int64_t pr = idx / half_n;
    const int vl = (int)(pr % kpairs);
    const int64_t image = pr / kpairs;
    const int vc = (int)(image % nvc);
    const int uc = (int)((image / nvc) % nuc);
    const int64_t plane = image / (nvc * nuc);
    const int u = uc * Uc + ul, v = vc * Vc + vl;
    float2 p = make_float2(0.f, 0.f);                                         // padding entries are written as zeros
    if (ul < Uc && vl < Vc && u < U && v < Vn) {
        const int64_t n = plane / 3;
        const int comp = (int)(plane - n * 3);
        p = P[n * ldP + (int64_t)comp * U * Vn + (int64_t)v * U + u];
    }
    const size_t img_bytes = (size_t)N1 * K1p * 2;
    ts_image_store(img + (size_t)image * 2 * img_bytes, img_bytes, N1, ul, vl, p.x, p.y);
}

// Exterior field straight into the spectrum images (eq. 9, then eq. 10 by the synthesis kernel): thread =
// (z plane, image (uc, vc), vl, ul) evaluates p_comp(s_m, z) = p_inc G[s_z, z_inc, z] + p_face G[-/+ s_z, z_face, z] for the
// three components (one s_z, two propagators) and writes their image entries; P never goes to memory.
struct TsExterior {
    int side;
    double lam_over_X, lam_over_Y, inv_lambda, n_re, n_im, z_face, z_inc;
    const float2* p_face;
    const float2* p_inc;
};

__global__ void k_tc_synth_exterior_images(int U, int Vn, int Uc, int Vc, int nuc, int nvc, int K1p, int N1, int Fz,
                                           const TsExterior e, const double* __restrict__ z, uint8_t* __restrict__ img,
                                           int* __restrict__ sched, int n_sched)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // (plane n, uc, vc, vl, ul), ul fastest
    for (int64_t i = idx; i < n_sched; i += (int64_t)gridDim.x * blockDim.x) sched[i] = 0;
    const int half_n = N1 / 2, kpairs = K1p / 2;
    if (idx >= (int64_t)Fz * nuc * nvc * half_n * kpairs) return;
    const int ul = (int)(idx % half_n);
    int64_t rest = idx / half_n;
    const int vl = (int)(rest % kpairs);
    rest /= kpairs;
    const int vc = (int)(rest % nvc);
    rest /= nvc;
    const int uc = (int)(rest % nuc);
    const int64_t n = rest / nuc;
    const int u = uc * Uc + ul, v = vc * Vc + vl;
    const bool real = ul < Uc && vl < Vc && u < U && v < Vn;
    float2 p[3] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};      // padding entries: zeros
    if (real) {
        const int m = v * U + u;
        const double sx = (double)(u - U / 2) * e.lam_over_X, sy = (double)(v - Vn / 2) * e.lam_over_Y;
        const double2 sz = ext_sz(e.n_re, e.n_im, sx, sy);
        const double zi = z[n];
        const double2 gf = e.side == SCW_SIDE_BELOW ? sz : make_double2(-sz.x, -sz.y);
        const double2 wf = ext_green(gf, (zi - e.z_face) * e.inv_lambda);
        const bool inc = e.side == SCW_SIDE_ABOVE && e.p_inc != nullptr;
        const double2 wi = inc ? ext_green(sz, (zi - e.z_inc) * e.inv_lambda) : make_double2(0.0, 0.0);
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            const float2 a = e.p_face[3 * m + comp];
            double er = (double)a.x * wf.x - (double)a.y * wf.y, ei = (double)a.x * wf.y + (double)a.y * wf.x;
            if (inc) {
                const float2 b = e.p_inc[3 * m + comp];
                er += (double)b.x * wi.x - (double)b.y * wi.y;
                ei += (double)b.x * wi.y + (double)b.y * wi.x;
            }
            p[comp] = make_float2((float)er, (float)ei);
        }
    }
    const size_t img_bytes = (size_t)N1 * K1p * 2;
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
        const int64_t image = ((n * 3 + comp) * nuc + uc) * nvc + vc;
        ts_image_store(img + (size_t)image * 2 * img_bytes, img_bytes, N1, ul, vl, p[comp].x, p[comp].y);
    }
}

// ---- main kernel ------------------------------------------------------------------------------------
// Three-product bf16 GEMM over K = Kp: D (+)= Ahi*Bhi + Ahi*Blo + Alo*Bhi.  `acc` = accumulate onto D.  The descriptors of
// k step s are the step-0 descriptors plus a constant (the address field is in 16-byte units), so the issuing
// thread spends two 64-bit adds per MMA instead of rebuilding descriptors.
// SS form: both operands are K-major shared-memory images (LBO a_lbo / b_lbo bytes between the 8-wide k chunks).
__device__ __forceinline__ void ts_mma3_ss(uint32_t d_tmem, uint32_t a_hi, uint32_t a_lo, uint32_t a_lbo, uint32_t b_hi,
                                           uint32_t b_lo, uint32_t b_lbo, int Kp, uint32_t idesc, uint32_t acc)
{
    uint64_t da_hi = umma_desc(a_hi, a_lbo, 128), da_lo = umma_desc(a_lo, a_lbo, 128);
    uint64_t db_hi = umma_desc(b_hi, b_lbo, 128), db_lo = umma_desc(b_lo, b_lbo, 128);
    const uint64_t a_step = (uint64_t)((2 * a_lbo) >> 4), b_step = (uint64_t)((2 * b_lbo) >> 4);
    for (int s = 0; s < Kp / 16; ++s) {
        umma_bf16(d_tmem, da_lo, db_hi, idesc, acc);
        acc = 1;
        umma_bf16(d_tmem, da_hi, db_lo, idesc, 1);
        umma_bf16(d_tmem, da_hi, db_hi, idesc, 1);
        da_hi += a_step; da_lo += a_step; db_hi += b_step; db_lo += b_step;
    }
}
// TS form: A is a TMEM block (column c = bf16 pair k = 2c, 2c+1; hi at ta_hi, lo at ta_lo), B a shared-memory image.
__device__ __forceinline__ void ts_mma3_ts(uint32_t d_tmem, uint32_t ta_hi, uint32_t ta_lo, uint32_t b_hi, uint32_t b_lo,
                                           uint32_t b_lbo, int Kp, uint32_t idesc, uint32_t acc)
{
    uint64_t db_hi = umma_desc(b_hi, b_lbo, 128), db_lo = umma_desc(b_lo, b_lbo, 128);
    const uint64_t b_step = (uint64_t)((2 * b_lbo) >> 4);
    for (int s = 0; s < Kp / 16; ++s) {
        umma_bf16_ts(d_tmem, ta_lo, db_hi, idesc, acc);
        acc = 1;
        umma_bf16_ts(d_tmem, ta_hi, db_lo, idesc, 1);
        umma_bf16_ts(d_tmem, ta_hi, db_hi, idesc, 1);
        ta_hi += 8; ta_lo += 8; db_hi += b_step; db_lo += b_step;
    }
}

template <bool INTENSITY>
__global__ void __launch_bounds__(TS_THREADS, 1) k_tc_synth(const __grid_constant__ TsParams p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int K1p = p.K1p, K2p = p.K2p, N1 = p.K2p, nuc = p.nuc, nvc = p.nvc;
    const uint32_t a1_img = TS_TILE * K1p * 2;                                 // bytes of one (hi or lo) image
    const uint32_t b1_img = (uint32_t)N1 * K1p * 2, b2_img = TS_TILE * K2p * 2;
    uint8_t* sA1 = smem;                              // nvc x (hi | lo)
    uint8_t* sB1 = sA1 + (size_t)nvc * 2 * a1_img;    // 2 stages x (hi | lo)
    uint8_t* sB2 = sB1 + 4 * b1_img;                  // b2_stages x 2 halves x (hi | lo)
    uint64_t* bars = reinterpret_cast<uint64_t*>(sB2 + (size_t)p.b2_stages * 4 * b2_img);
    uint64_t* tw_full = bars;            // [1]
    uint64_t* b1_full = bars + 1;        // [2]
    uint64_t* b1_empty = bars + 3;       // [2]
    uint64_t* d1_full = bars + 5;        // [1]
    uint64_t* d1_empty = bars + 6;       // [1]
    uint64_t* b2_full = bars + 7;        // [2]
    uint64_t* b2_empty = bars + 9;       // [2]
    uint64_t* d2_full = bars + 11;       // [2]
    uint64_t* d2_empty = bars + 13;      // [2]
    uint64_t* sched_full = bars + 15;    // [8] plane ids handed from the loader to the other roles
    int* s_plane = reinterpret_cast<int*>(bars + 23);               // [8]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 27);
    uint64_t* a2_full = bars + 28;       // [1] x twiddles are in TMEM (converter warps -> MMA warp)
    uint64_t* b2_full_s1 = bars + 29;    // [2] second B2 stage (b2_stages == 2)
    uint64_t* b2_empty_s1 = bars + 31;   // [2]
    const int b2s = p.b2_stages;

    if (tid == 0) {
        if (blockIdx.x == 0 && p.tl_slot) *p.tl_slot = 0ull;   // this launch's timeline slot (atomicMax at the CTAs' exits)
        mbar_init(tw_full, 1);
        mbar_init(a2_full, 8);
        for (int s = 0; s < 8; ++s) mbar_init(&sched_full[s], 1);
        for (int s = 0; s < 2; ++s) {
            mbar_init(&b1_full[s], 1);
            mbar_init(&b1_empty[s], 1);
            mbar_init(&b2_full[s], 4);
            mbar_init(&b2_empty[s], 1);
            mbar_init(&b2_full_s1[s], 4);
            mbar_init(&b2_empty_s1[s], 1);
            mbar_init(&d2_full[s], 1);
            mbar_init(&d2_empty[s], 8);
        }
        mbar_init(d1_full, 1);
        mbar_init(d1_empty, 8);
        mbar_fence_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, TS_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const uint32_t a2_col = TS_D1_COL + N1;                    // A2 chunk uc: hi at a2_col + uc*K2p, lo K2p/2 columns on

    // This CTA's tile pair.  Its planes are handed out dynamically: the CTAs of a pair draw plane ids from a shared
    // counter (the kernel is HBM-write-bound and the SMs do not all run at the same pace, a static split leaves a tail).
    // The loader draws the id and publishes it through an 8-deep ring (the loader is never more than 6 planes ahead of
    // the epilogue); id -1 ends every role.  Item = (plane, u chunk).
    const int pair = p.pair0 + (int)blockIdx.x % p.npairs;
    const int tx = pair % p.tiles_x, ty = pair / p.tiles_x;
    auto sched_get = [&](int nl) -> int {
        mbar_wait(&sched_full[nl & 7], (nl >> 3) & 1);
        return *reinterpret_cast<volatile int*>(&s_plane[nl & 7]);
    };

    // A2 (the x twiddles of this tile, every u chunk) goes to TMEM once: the converter warp pair of lane quarter q
    // writes rows 32q..32q+31, warp kg = 0 the hi words, kg = 1 the lo words
    if (warp >= 2 && warp < 10) {
        const int q = warp & 3, kg = (warp - 2) >> 2;
        const int half = K2p / 2;
        for (int uc = 0; uc < nuc; ++uc) {
            const uint4* src = reinterpret_cast<const uint4*>(p.A2 + (((size_t)tx * nuc + uc) * TS_TILE + 32 * q + lane) * K2p +
                                                              kg * half);
            const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + a2_col + uc * K2p + kg * half;
            for (int c8 = 0; c8 < half / 8; ++c8) {
                const uint4 v0 = __ldcg(src + 2 * c8), v1 = __ldcg(src + 2 * c8 + 1);      // L2: this runs before pdl_wait()
                const uint32_t r[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
                tmem_st8(taddr + 8 * c8, r);
            }
        }
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(a2_full);           // only GEMM2 needs A2: the other roles do not wait for it
    }

    // Everything above (barriers, TMEM, the x twiddles -- written by the twiddle kernel, which the assembly before this
    // kernel has already waited for) predates the assembly that feeds this kernel; the spectrum images and the plane
    // counters are its output: wait for it here (PDL), then let the next kernel's prologue start.
    pdl_wait();
    pdl_launch_dependents();

    if (warp == 0) {
        // ===== loader: draws the planes; y twiddle images once, then the nuc*nvc spectrum images of every plane =====
        if (lane == 0) {
            int q = 0, g = 0;
            for (int nl = 0;; ++nl) {
                const int c = nl % p.group;                 // a drawn unit is `group` consecutive planes
                if (c == 0) g = atomicAdd(&p.sched[pair], 1);
                int plane = g * p.group + c;
                if (plane >= p.planes) plane = -1;
                *reinterpret_cast<volatile int*>(&s_plane[nl & 7]) = plane;
                mbar_arrive(&sched_full[nl & 7]);
                if (plane < 0) break;
                if (nl == 0) {
                    mbar_expect_tx(tw_full, nvc * 2 * a1_img);
                    bulk_g2s(sA1, p.A1 + (size_t)ty * nvc * 2 * a1_img, nvc * 2 * a1_img, tw_full);
                }
                for (int uc = 0; uc < nuc; ++uc)
                    for (int vc = 0; vc < nvc; ++vc, ++q) {
                        const int s = q & 1;
                        mbar_wait(&b1_empty[s], ((q >> 1) & 1) ^ 1);
                        mbar_expect_tx(&b1_full[s], 2 * b1_img);
                        bulk_g2s(sB1 + (size_t)s * 2 * b1_img, p.B1 + (((size_t)plane * nuc + uc) * nvc + vc) * 2 * b1_img,
                                 2 * b1_img, &b1_full[s]);
                    }
            }
        }
    } else if (warp == 1 || warp == TS_GEMM1_WARP) {
        // ===== MMA issuers: GEMM1 (warp 18) and GEMM2 (warp 1) are issued by different warps.  One thread needs ~100 cycles
        // per tcgen05.mma it issues (descriptor arithmetic, the instruction itself, the barriers around a GEMM) and a plane
        // takes 27 (17 x 17 frequencies) to 45 (33 x 33) of them: with a single issuer the detector mode, which stores
        // almost nothing, ran at the issue rate (2.1 us per plane), not at the tensor pipe's.  The two chains only meet
        // through D1 (d1_full / d1_empty via the converters), which the mbarriers already order.  The whole warp runs the
        // loop (warp-uniform control flow), one elected lane issues. =====
        if (sched_get(0) >= 0) {
            const uint32_t idesc1 = umma_idesc_bf16(TS_TILE, N1, false, true);    // B1 (spectrum images) is MN-major
            const uint32_t idesc2 = umma_idesc_bf16(TS_TILE, TS_TILE);
            const uint32_t a1 = smem_u32(sA1), b1 = smem_u32(sB1), b2 = smem_u32(sB2);
            const uint32_t d1 = tmem_base + TS_D1_COL;
            auto issue_gemm1 = [&](int i) {            // D1 = sum over the v chunks of item i
                for (int vc = 0; vc < nvc; ++vc) {
                    const int q = i * nvc + vc, s = q & 1;
                    mbar_wait(&b1_full[s], (q >> 1) & 1);
                    if (vc == 0 && i > 0) mbar_wait(d1_empty, (i - 1) & 1);
                    tc_fence_after();
                    if (elect_one()) {
                        ts_mma3_ss(d1, a1 + vc * 2 * a1_img, a1 + vc * 2 * a1_img + a1_img, 2048, b1 + s * 2 * b1_img,
                                   b1 + s * 2 * b1_img + b1_img, (uint32_t)N1 * 16, K1p, idesc1, vc > 0 ? 1u : 0u);
                        umma_commit(&b1_empty[s]);
                        if (vc == nvc - 1) umma_commit(d1_full);
                    }
                    __syncwarp();
                }
            };
            auto issue_gemm2 = [&](int i, int h) {     // D2[h] (+)= A2[uc] B2[h]; complete after the last u chunk
                const int n = i / nuc, uc = i - n * nuc;
                if (i == 0 && h == 0) mbar_wait(a2_full, 0);
                const int st = b2s == 2 ? (i & 1) : 0;                    // B2 stage of this item and how often it was used
                const int su = b2s == 2 ? (i >> 1) : i;
                mbar_wait(st ? &b2_full_s1[h] : &b2_full[h], su & 1);
                const int hb = p.d2_single ? 0 : h;                       // D2 buffer of this half, and how often it was used
                const int use = p.d2_single ? 2 * n + h : n;
                if (uc == 0) mbar_wait(&d2_empty[hb], (use & 1) ^ 1);
                tc_fence_after();
                const uint32_t ta = tmem_base + a2_col + uc * K2p;
                if (elect_one()) {
                    const uint32_t b2h = b2 + (uint32_t)(st * 4 + h * 2) * b2_img;
                    ts_mma3_ts(tmem_base + TS_D2_COL + hb * TS_TILE, ta, ta + K2p / 2, b2h, b2h + b2_img, 2048, K2p, idesc2,
                               uc > 0 ? 1u : 0u);
                    umma_commit(st ? &b2_empty_s1[h] : &b2_empty[h]);
                    if (uc == nuc - 1) umma_commit(&d2_full[hb]);
                }
                __syncwarp();
            };
            if (warp == TS_GEMM1_WARP) mbar_wait(tw_full, 0);              // the y twiddle images (A1) are in shared memory
            for (int i = 0;; ++i) {                                        // item i = (plane n, u chunk uc)
                const int n = i / nuc, uc = i - n * nuc;
                if (uc == 0 && i > 0 && sched_get(n) < 0) break;
                if (warp == TS_GEMM1_WARP) {
                    issue_gemm1(i);
                } else {
                    issue_gemm2(i, 0);
                    issue_gemm2(i, 1);
                }
            }
        }
    } else if (warp < 10) {
        // ===== converters: D1 row y (TMEM) -> B2 rows (y,Re), (y,Im) as bf16 hi/lo.  Two warps per TMEM lane
        // quarter: warp kg = 0/1 takes the even/odd 8-column chunks of the row. =====
        const int q = warp & 3;                      // TMEM lane quarter: y = 32q + lane
        const int kg = (warp - 2) >> 2;              // chunk parity handled by this warp
        const int h = q >> 1;                        // which half of the tile this y belongs to
        const int yy = 32 * (q & 1) + lane;          // y within the half
        uint8_t* row0 = sB2 + (size_t)h * 2 * b2_img + yy * 32;
        const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + TS_D1_COL;
        const int nchunks = K2p / 8;                 // <= 10
        for (int n = 0;; ++n) {                      // n = item (plane, u chunk)
            if (n % nuc == 0 && sched_get(n / nuc) < 0) break;
            mbar_wait(d1_full, n & 1);
            tc_fence_after();
            uint32_t t[5][8];
#pragma unroll
            for (int i = 0; i < 5; ++i)
                if (2 * i + kg < nchunks) tmem_ld8_raw(taddr + 8 * (2 * i + kg), t[i]);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(d1_empty);    // D1 may be overwritten by the next plane's GEMM1
            const int st = b2s == 2 ? (n & 1) : 0, su = b2s == 2 ? (n >> 1) : n;
            uint8_t* row = row0 + (size_t)st * 4 * b2_img;
            mbar_wait(st ? &b2_empty_s1[h] : &b2_empty[h], (su & 1) ^ 1);
#pragma unroll
            for (int i = 0; i < 5; ++i) {
                const int c = 2 * i + kg;
                if (c < nchunks) {
                    float f[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(t[i][e]);   // (Tr0, Ti0, ..., Tr3, Ti3)
                    // one split per (T_r, T_i) pair; row (y,Re) holds (T_r, -T_i): sign flip of the upper half (round to
                    // nearest is odd, so hi/lo of -t are -hi/-lo of t); row (y,Im) holds (T_i, T_r): the halves swapped.
                    // The conversion instruction is the converters' scarce resource (16 lanes/clk/SM).
                    uint32_t H[4], Lw[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) split_bf16x2(f[2 * k], f[2 * k + 1], H[k], Lw[k]);
                    const uint4 re_hi = make_uint4(H[0] ^ 0x80000000u, H[1] ^ 0x80000000u, H[2] ^ 0x80000000u, H[3] ^ 0x80000000u);
                    const uint4 re_lo = make_uint4(Lw[0] ^ 0x80000000u, Lw[1] ^ 0x80000000u, Lw[2] ^ 0x80000000u, Lw[3] ^ 0x80000000u);
                    const uint4 im_hi = make_uint4(__byte_perm(H[0], 0, 0x1032), __byte_perm(H[1], 0, 0x1032),
                                                   __byte_perm(H[2], 0, 0x1032), __byte_perm(H[3], 0, 0x1032));
                    const uint4 im_lo = make_uint4(__byte_perm(Lw[0], 0, 0x1032), __byte_perm(Lw[1], 0, 0x1032),
                                                   __byte_perm(Lw[2], 0, 0x1032), __byte_perm(Lw[3], 0, 0x1032));
                    uint8_t* dst = row + (size_t)c * 2048;
                    *reinterpret_cast<uint4*>(dst) = re_hi;
                    *reinterpret_cast<uint4*>(dst + 16) = im_hi;
                    *reinterpret_cast<uint4*>(dst + b2_img) = re_lo;
                    *reinterpret_cast<uint4*>(dst + b2_img + 16) = im_lo;
                }
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(st ? &b2_full_s1[h] : &b2_full[h]);
        }
    } else {
        // ===== epilogue: D2 (lane = x, columns = (y, Re/Im)) -> E.  Two warps per lane quarter, 32 y each. =====
        const int q = warp & 3;
        const int cg = (warp - 10) >> 2;             // which 32-y group of the half
        const int64_t x = (int64_t)tx * TS_TILE + 32 * q + lane;
        const bool x_ok = x < p.Nx;
        for (int n = 0;; ++n) {
            const int gplane = sched_get(n);
            if (gplane < 0) break;
            const int inst = gplane / p.planes_per_inst;
            const int plane = gplane - inst * p.planes_per_inst;
            const int64_t zi = plane / 3;
            const int comp = plane - (int)zi * 3;
            float2* const Einst = p.E[inst];
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {
                const int64_t y0 = (int64_t)ty * TS_TILE + 64 * h + 32 * cg;
                const int ny = (int)min((int64_t)32, p.Ny - y0);   // may be <= 0
                const int hb = p.d2_single ? 0 : h;
                mbar_wait(&d2_full[hb], (p.d2_single ? 2 * n + h : n) & 1);
                tc_fence_after();
                const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + TS_D2_COL + hb * TS_TILE + 64 * cg;
                if (INTENSITY) {
                    // detector: |E_comp|^2 per sample, then (want_I) I = |E_x|^2 + |E_y|^2 + |E_z|^2 and / or (s_part) the
                    // sum over a window of the plane.  D2[h] is released as soon as it is in registers, like the complex
                    // path.  For I the three components of a z plane come to this CTA in order (group = 3) and every
                    // (x, y) belongs to one thread: the running sum lives in 128 TMEM columns (lane = x, column = y) at
                    // p.acc_col -- spare columns behind A2 (U <= 32), or the second half of D2 when D2 is single-buffered
                    // (d2_single, 32 < U <= 40) -- and only the third component writes the output; with two u chunks
                    // (U > 40) GEMM2 accumulates both y halves across the chunks, D2 cannot shrink and the sum is kept in
                    // the output itself (read-modify-write through L2).
                    const uint32_t acc = tmem_base + ((uint32_t)(32 * q) << 16) + p.acc_col + h * 64 + 32 * cg;
                    float m2[32];
                    {
                        uint32_t v[2][32];
                        tmem_ld32_raw(taddr, v[0]);
                        tmem_ld32_raw(taddr + 32, v[1]);
                        tmem_ld_wait();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&d2_empty[hb]); // D2 is in registers now
#pragma unroll
                        for (int e = 0; e < 32; ++e) {
                            const float re = __uint_as_float(v[e >> 4][(2 * e) & 31]), im = __uint_as_float(v[e >> 4][(2 * e + 1) & 31]);
                            m2[e] = re * re + im * im;
                        }
                    }
                    if (p.s_part) {                                // window sum of this warp's 32 x 32 patch, fixed order
                        // bit e of ymask: (x, y0 + e) lies in the window (branch-free selects: a branch per sample costs more
                        // than the whole epilogue)
                        const int lo = (int)max((int64_t)0, (int64_t)p.win_y0 - y0), hi = (int)min((int64_t)32, (int64_t)p.win_y1 - y0);
                        uint32_t ymask = 0u;
                        if (x >= p.win_x0 && x < p.win_x1 && hi > lo)
                            ymask = (hi >= 32 ? 0xffffffffu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
                        float ws = 0.f;
#pragma unroll
                        for (int e = 0; e < 32; ++e) ws += ((ymask >> e) & 1u) ? m2[e] : 0.f;
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) ws += __shfl_xor_sync(0xffffffffu, ws, o);
                        if (lane == 0)
                            p.s_part[((size_t)gplane * (p.tiles_x * p.tiles_y) + pair) * 16 + h * 8 + cg * 4 + q] = ws;
                    }
                    if (p.want_I) {
                        float* io = reinterpret_cast<float*>(Einst) + zi * p.s_z + x * p.s_x + y0 * p.s_y;
                        if (p.acc_col) {
                            if (comp > 0) {
                                float a[2][16];
                                tmem_st_wait();                    // the previous component's sums have landed
                                tmem_ld16(acc, a[0]);
                                tmem_ld16(acc + 16, a[1]);
                                tmem_ld_wait();
#pragma unroll
                                for (int e = 0; e < 32; ++e) m2[e] += a[e >> 4][e & 15];
                            }
                            if (comp < 2) {
                                uint32_t w0[16], w1[16];
#pragma unroll
                                for (int e = 0; e < 16; ++e) {
                                    w0[e] = __float_as_uint(m2[e]);
                                    w1[e] = __float_as_uint(m2[16 + e]);
                                }
                                tmem_st16(acc, w0);
                                tmem_st16(acc + 16, w1);
                            } else if (x_ok) {
#pragma unroll
                                for (int e = 0; e < 32; ++e)
                                    if (e < ny) __stcg(io + e * p.s_y, m2[e]);
                            }
                        } else if (x_ok) {                         // no TMEM room (two u chunks, U > 40): sum kept in the output
#pragma unroll
                            for (int e = 0; e < 32; ++e) {
                                if (e < ny) {
                                    const float prev = comp > 0 ? __ldcg(io + e * p.s_y) : 0.f;
                                    __stcg(io + e * p.s_y, prev + m2[e]);
                                }
                            }
                        }
                    }
                } else {
                    uint32_t v[2][32];
                    tmem_ld32_raw(taddr, v[0]);
                    tmem_ld32_raw(taddr + 32, v[1]);
                    tmem_ld_wait();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&d2_empty[hb]);     // D2[h] is in registers now
                    float2* out = Einst + comp * p.s_comp + zi * p.s_z + x * p.s_x + y0 * p.s_y;
                    if (x_ok) {
#pragma unroll
                        for (int e = 0; e < 32; ++e) {
                            if (e < ny) {
                                const float2 val = make_float2(__uint_as_float(v[e >> 4][(2 * e) & 31]),
                                                               __uint_as_float(v[e >> 4][(2 * e + 1) & 31]));
                                __stcs(out + e * p.s_y, val);      // written once, never re-read here: evict-first
                            }
                        }
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, TS_TMEM_COLS);
    if (tid == 0 && p.tl_slot) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        atomicMax(p.tl_slot, t);
    }
}

// Window sums: S[inst][n] = sum over the three components, the output tiles and the 16 warp patches of a tile, in a fixed
// order (deterministic), of the partial sums the detector epilogue left in s_part.
__global__ void __launch_bounds__(128) k_tc_synth_wsum(int n_inst, int Fz, int tiles, const float* __restrict__ s_part,
                                                       const TsWsumOut out)
{
    const int idx = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;      // one warp per (inst, n)
    if (idx >= n_inst * Fz) return;
    const int inst = idx / Fz, n = idx - inst * Fz;
    const int cnt = 3 * tiles * 16;
    const float* src = s_part + (size_t)idx * cnt;                    // plane (inst*Fz + n)*3 + comp, contiguous over comp
    float acc = 0.f;
    for (int i = lane; i < cnt; i += 32) acc += src[i];               // fixed order per lane, then a fixed tree
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) out.S[inst][n] = acc;
}

// ---- host side -------------------------------------------------------------------------------------
struct TsPlan {
    TsChunks cu, cv;          // frequency chunks along u (GEMM2's K) and v (GEMM1's K)
    int K1p, K2p, tiles_x, tiles_y;
    size_t a1_bytes, a2_bytes, sched_bytes, b1_bytes, smem_bytes;
    int b2_stages;
};

static TsPlan ts_plan(int U, int Vn, int64_t Fz, int64_t Nx, int64_t Ny)
{
    TsPlan pl;
    pl.cu = ts_chunks(U);
    pl.cv = ts_chunks(Vn);
    pl.K1p = pl.cv.Kp;
    pl.K2p = pl.cu.Kp;
    pl.tiles_x = (int)((Nx + TS_TILE - 1) / TS_TILE);
    pl.tiles_y = (int)((Ny + TS_TILE - 1) / TS_TILE);
    pl.a1_bytes = align_up((size_t)pl.tiles_y * pl.cv.n * 2 * TS_TILE * pl.K1p * 2);
    pl.a2_bytes = align_up((size_t)pl.tiles_x * pl.cu.n * TS_TILE * pl.K2p * 4);
    pl.sched_bytes = align_up((size_t)pl.tiles_x * pl.tiles_y * sizeof(int));
    pl.b1_bytes = align_up((size_t)Fz * 3 * pl.cu.n * pl.cv.n * 2 * pl.K2p * pl.K1p * 2);
    const size_t b2_bytes = (size_t)4 * TS_TILE * pl.K2p * 2;                  // one B2 buffer: 2 halves x (hi | lo)
    pl.smem_bytes = (size_t)pl.cv.n * 2 * TS_TILE * pl.K1p * 2 + (size_t)4 * pl.K2p * pl.K1p * 2 + b2_bytes + 512;
    // a second B2 buffer when it fits (up to 24 frequencies along u): the converters then split plane i + 1 while GEMM2 still
    // reads plane i (with one buffer GEMM2 -> converters -> GEMM2 is a serial chain: 2.1 us per plane at 17 x 17 frequencies
    // against 1.1 us of MMA issue)
    pl.b2_stages = pl.smem_bytes + b2_bytes <= 227 * 1024 ? 2 : 1;
    if (pl.b2_stages == 2) pl.smem_bytes += b2_bytes;
    return pl;
}

// up to TS_FMAX frequencies per axis: TMEM holds D2 (256 columns), D1 (K2p) and A2 (K2p per u chunk)
bool tc_synth_supported(int dtype, int U, int Vn)
{
    if (dtype != SCW_C64 || U > TS_FMAX || Vn > TS_FMAX) return false;
    const TsPlan pl = ts_plan(U, Vn, 1, 1, 1);
    return TS_D1_COL + pl.K2p * (1 + pl.cu.n) <= TS_TMEM_COLS && pl.smem_bytes <= 227 * 1024;
}

size_t tc_synth_twiddle_bytes(int U, int Vn, int64_t Nx, int64_t Ny)
{
    const TsPlan pl = ts_plan(U, Vn, 1, Nx, Ny);
    return pl.a1_bytes + pl.a2_bytes + pl.sched_bytes;      // y images | x operand rows | plane counters
}

size_t tc_synth_scratch(int U, int Vn, int64_t Fz) { return ts_plan(U, Vn, Fz, 1, 1).b1_bytes; }

void launch_tc_synth_twiddles(scw_ctx* ctx, int U, int Vn, double X, double Y, int64_t Nx, const double* x, int64_t Ny,
                              const double* y, void* tw, int* zero, size_t n_zero)
{
    const TsPlan pl = ts_plan(U, Vn, 1, Nx, Ny);
    uint8_t* A1 = static_cast<uint8_t*>(tw);
    uint8_t* A2 = A1 + pl.a1_bytes;
    const TwAxis ay{Vn, pl.cv.n, pl.cv.len, pl.K1p, pl.tiles_y, Ny, y, 1.0 / Y, A1};
    const TwAxis ax{U, pl.cu.n, pl.cu.len, pl.K2p, pl.tiles_x, Nx, x, 1.0 / X, A2};
    const int64_t ny = (int64_t)pl.tiles_y * pl.cv.n * TS_TILE * (pl.K1p / 2);
    const int64_t nx = (int64_t)pl.tiles_x * pl.cu.n * TS_TILE * (pl.K2p / 2);
    const int by = (int)((ny + 255) / 256), bx = (int)((nx + 255) / 256);
    KernelScope ks(ctx, KC_TWIDDLES);
    k_tc_synth_twiddles<<<by + bx, 256, 0, ctx->stream>>>(ay, ax, by, zero, zero ? n_zero : 0);
}


int tc_synth_max_group() { return TS_MAX_INST; }

static int* ts_sched(const TsPlan& pl, const void* tw)
{
    return reinterpret_cast<int*>(static_cast<uint8_t*>(const_cast<void*>(tw)) + pl.a1_bytes + pl.a2_bytes);
}

// The synthesis launches proper: B1 holds the spectrum images of all n_inst*Fz*3 planes.
static void ts_launch_main(scw_ctx* ctx, const TsPlan& pl, int64_t Fz, int n_inst, const uint8_t* B1, int64_t Nx,
                           int64_t Ny, const void* tw, void* const* E, const int64_t strides[4], const TcDetector* det)
{
    const bool intensity = det != nullptr;
    const bool want_I = intensity && det->I != nullptr;
    static thread_local TsParams p;
    const int planes = (int)(Fz * 3 * n_inst);
    p.A1 = static_cast<const uint8_t*>(tw);
    p.A2 = reinterpret_cast<const uint32_t*>(p.A1 + pl.a1_bytes);
    p.B1 = B1;
    p.sched = ts_sched(pl, tw);
    for (int i = 0; i < n_inst; ++i) p.E[i] = static_cast<float2*>(intensity ? (want_I ? det->I[i] : nullptr) : E[i]);
    p.s_comp = strides[0];
    p.s_z = strides[1];
    p.s_y = strides[2];
    p.s_x = strides[3];
    p.Nx = Nx;
    p.Ny = Ny;
    p.planes = planes;
    p.planes_per_inst = (int)(Fz * 3);
    p.K1p = pl.K1p;
    p.K2p = pl.K2p;
    p.nuc = pl.cu.n;
    p.nvc = pl.cv.n;
    p.want_I = want_I ? 1 : 0;
    p.group = want_I ? 3 : 1;
    {   // detector accumulators (128 columns): behind D2 | D1 | A2 when they fit (U <= 32); else D2 shrinks to one
        // 128-column buffer shared by the two y halves and the sum takes the columns of its second half
        const int used = TS_D1_COL + pl.K2p * (1 + pl.cu.n);
        const bool fits = used + 128 <= TS_TMEM_COLS;
        p.d2_single = (want_I && !fits && pl.cu.n == 1) ? 1 : 0;
        p.acc_col = !want_I ? 0 : (fits ? used : (p.d2_single ? TS_TILE : 0));
    }
    p.b2_stages = pl.b2_stages;
    p.s_part = (intensity && det->S) ? static_cast<float*>(det->s_part) : nullptr;
    if (intensity) {
        p.win_x0 = (int)det->win[0]; p.win_x1 = (int)det->win[1]; p.win_y0 = (int)det->win[2]; p.win_y1 = (int)det->win[3];
    }
    const size_t smem_bytes = pl.smem_bytes;
    p.tiles_x = pl.tiles_x;
    p.tiles_y = pl.tiles_y;
    const int total_pairs = pl.tiles_x * pl.tiles_y;
    if (intensity) cudaFuncSetAttribute(k_tc_synth<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    else cudaFuncSetAttribute(k_tc_synth<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    for (int pair0 = 0; pair0 < total_pairs; pair0 += ctx->sm_count) {
        p.pair0 = pair0;
        p.npairs = total_pairs - pair0 < ctx->sm_count ? total_pairs - pair0 : ctx->sm_count;
        int per_pair = ctx->sm_count / p.npairs;
        if (per_pair > planes) per_pair = planes;
        KernelScope ks(ctx, KC_SYNTH_TC);
        p.tl_slot = tl_next(ctx, KC_SYNTH_TC);
        if (intensity) launch_pdl(k_tc_synth<true>, dim3(p.npairs * per_pair), dim3(TS_THREADS), smem_bytes, ctx->stream, p);
        else launch_pdl(k_tc_synth<false>, dim3(p.npairs * per_pair), dim3(TS_THREADS), smem_bytes, ctx->stream, p);
    }
    if (p.s_part) {
        TsWsumOut out;
        for (int i = 0; i < n_inst; ++i) out.S[i] = static_cast<float*>(det->S[i]);
        KernelScope ks(ctx, KC_MISC);
        const int n = n_inst * (int)Fz;
        k_tc_synth_wsum<<<(n + 3) / 4, 128, 0, ctx->stream>>>(n_inst, (int)Fz, total_pairs, p.s_part, out);
    }
}

size_t tc_synth_wsum_bytes(int64_t planes_z, int64_t Nx, int64_t Ny)
{
    const int64_t tiles = ((Nx + TS_TILE - 1) / TS_TILE) * ((Ny + TS_TILE - 1) / TS_TILE);
    return align_up((size_t)planes_z * 3 * tiles * 16 * sizeof(float));
}

// n_inst <= TS_MAX_INST instances with the same Fz whose spectra are stored back to back
// (P_all is one column-major [ldP x n_inst*Fz] matrix): one image pre-kernel + one synthesis launch.
void launch_tc_synth_group(scw_ctx* ctx, int U, int Vn, int64_t Fz, int n_inst, const void* P_all, int64_t ldP,
                           int64_t Nx, int64_t Ny, const void* tw, void* const* E, const int64_t strides[4],
                           void* scratch, const TcDetector* det)
{
    const TsPlan pl = ts_plan(U, Vn, Fz * n_inst, Nx, Ny);
    const int planes = (int)(Fz * 3 * n_inst);
    uint8_t* B1 = static_cast<uint8_t*>(scratch);
    {
        KernelScope ks(ctx, KC_SYNTH_IMG);
        const int64_t n = (int64_t)planes * pl.cu.n * pl.cv.n * (pl.K2p / 2) * (pl.K1p / 2);
        k_tc_synth_pimage<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(U, Vn, pl.cu.len, pl.cv.len, pl.cu.n, pl.cv.n,
                                                                                pl.K1p, pl.K2p, planes, (const float2*)P_all,
                                                                                ldP, B1, ts_sched(pl, tw),
                                                                                pl.tiles_x * pl.tiles_y);
    }
    ts_launch_main(ctx, pl, Fz, n_inst, B1, Nx, Ny, tw, E, strides, det);
}

void tc_synth_image_plan(int U, int Vn, int64_t Nx, int64_t Ny, void* scratch, const void* tw, TcFixup* fix, int** sched,
                         int* n_sched)
{
    const TsPlan pl = ts_plan(U, Vn, 1, Nx, Ny);
    fix->mode = TC_FIX_IMAGES;
    fix->img = static_cast<uint8_t*>(scratch);
    fix->U = U;
    fix->Vn = Vn;
    fix->Uc = pl.cu.len;
    fix->Vc = pl.cv.len;
    fix->nuc = pl.cu.n;
    fix->nvc = pl.cv.n;
    fix->K1p = pl.K1p;
    fix->N1 = pl.K2p;
    *sched = ts_sched(pl, tw);
    *n_sched = pl.tiles_x * pl.tiles_y;
}

void launch_tc_synth_group_images(scw_ctx* ctx, int U, int Vn, int64_t Fz, int n_inst, int64_t Nx, int64_t Ny,
                                  const void* tw, void* const* E, const int64_t strides[4], void* scratch,
                                  const TcDetector* det)
{
    const TsPlan pl = ts_plan(U, Vn, Fz * n_inst, Nx, Ny);
    ts_launch_main(ctx, pl, Fz, n_inst, static_cast<const uint8_t*>(scratch), Nx, Ny, tw, E, strides, det);
}

// Exterior field on a grid in two launches: eq. 9 into the spectrum images, then the synthesis (eq. 10).
void launch_tc_synth_exterior(scw_ctx* ctx, const scw_exterior* e, int64_t Fz, const double* z, int64_t Nx, int64_t Ny,
                              const void* tw, void* E, const int64_t strides[4], void* scratch)
{
    const TsPlan pl = ts_plan(e->U, e->Vn, Fz, Nx, Ny);
    uint8_t* B1 = static_cast<uint8_t*>(scratch);
    TsExterior te;
    te.side = e->side;
    te.lam_over_X = e->lambda / e->X;
    te.lam_over_Y = e->lambda / e->Y;
    te.inv_lambda = 1.0 / e->lambda;
    te.n_re = e->n_re;
    te.n_im = e->n_im;
    te.z_face = e->z_face;
    te.z_inc = e->z_inc;
    te.p_face = static_cast<const float2*>(e->p_face);
    te.p_inc = static_cast<const float2*>(e->p_inc);
    {
        KernelScope ks(ctx, KC_EXTERIOR);
        const int64_t n = Fz * pl.cu.n * pl.cv.n * (pl.K2p / 2) * (pl.K1p / 2);
        k_tc_synth_exterior_images<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(
            e->U, e->Vn, pl.cu.len, pl.cv.len, pl.cu.n, pl.cv.n, pl.K1p, pl.K2p, (int)Fz, te, z, B1, ts_sched(pl, tw),
            pl.tiles_x * pl.tiles_y);
    }
    ts_launch_main(ctx, pl, Fz, 1, B1, Nx, Ny, tw, &E, strides, nullptr);
}

void launch_tc_synth(scw_ctx* ctx, int U, int Vn, int64_t Fz, const void* P, int64_t ldP, int64_t Nx, int64_t Ny,
                     const void* tw, void* E, const int64_t strides[4], void* scratch)
{
    launch_tc_synth_group(ctx, U, Vn, Fz, 1, P, ldP, Nx, Ny, tw, &E, strides, scratch, nullptr);
}

}  // namespace scw
