// Spectral assembly P = V . W on the 5th-gen tensor cores (tcgen05, accumulators in TMEM), complex64.
//
//   P[:, i] = V . (c o g(z_i))     (eq. 31 with the diag(alpha) factoring)
//
// Precision: fp32 operands are split in software into bf16 hi + lo (round to nearest) and three
// products hi*hi + hi*lo + lo*hi are accumulated in fp32 ("BF16x3", error ~1e-5 relative), because a
// single TF32/BF16 pass misses the 2e-4 bar.
// Complex on a real MMA: V (column-major interleaved complex) is viewed as a real matrix with 2R rows
// (rows 2r / 2r+1 = Re / Im of complex row r); the small operand is laid out as [W_r | W_i] so that one
// real GEMM yields all four real products, combined between adjacent TMEM lanes in the epilogue.
//
// Work decomposition ("stream-K"): the iteration space (n_tile, m_tile, k_block) is cut into equal
// contiguous spans, one per persistent CTA (one CTA per SM); every (CTA, tile) segment writes an fp32
// partial tile, k_tc_reduce sums the segments of each tile in a fixed order (deterministic).
//
// Warp roles (704 threads): warps 8-15 stream V from HBM with bulk async copies (cp.async.bulk, one per
// 512-byte column segment) into an fp32 staging ring that keeps 64-128 KB in flight per SM; warps 0-7
// split the staged fp32 into bf16 hi/lo and store K-major UMMA tiles; warp 16 fetches the pre-formatted
// W tiles with bulk async copies; warp 17 issues tcgen05.mma; warps 18-21 drain TMEM (tcgen05.ld),
// combine lanes with one shuffle per element and store the partial tile.
#include "scw_internal.h"
#include "scw_tc_common.cuh"

namespace scw {

using namespace tc;

constexpr int TA_BM = 128;                 // real rows per tile (= 64 complex rows)
constexpr int TA_BK = 64;                  // modes per pipeline stage
constexpr int TA_CONV_WARPS = 8;           // warp w converts k-chunk w (8 modes) of every stage
constexpr int TA_LOAD_WARPS = 8;           // V loader warps: 8 column copies each per stage
constexpr int TA_THREADS = (TA_CONV_WARPS + TA_LOAD_WARPS + 2 + 4) * 32;
constexpr int TA_D_COLS = 256;             // TMEM: two accumulators of N2 <= 128 columns
constexpr int TA_A_COL = TA_D_COLS;        // TMEM: A operand, per MMA stage 32 columns hi + 32 columns lo (bf16 pairs)
constexpr int TA_COL_PITCH = 528;          // fp32 staging: 512 B of a V column segment + 16 B alignment slack
constexpr int TA_STG_BYTES = TA_BK * TA_COL_PITCH;
constexpr int TA_MMA_STAGES = 2;
constexpr int TA_TMEM_COLS = 512;
constexpr int TA_SMEM_LIMIT = 226 * 1024;
constexpr int TA_V_LOADER = TA_CONV_WARPS, TA_W_LOADER = TA_V_LOADER + TA_LOAD_WARPS, TA_MMA_WARP = TA_W_LOADER + 1;

constexpr int TA_MAX_INST = 64;            // instances (layers x wavelengths) per grouped launch

#ifdef SCW_TS_DEBUG
__device__ long long g_ta_dbg[8192];
#define TA_MARK(slot) do { if (blockIdx.x == 0 && (slot) < 8192) g_ta_dbg[(slot)] = clock64(); } while (0)
__device__ long long g_ta_blk[4 * 256];
__device__ __forceinline__ long long ta_gtime() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TA_BLK(i) do { if (threadIdx.x == 0) { g_ta_blk[blockIdx.x * 4 + (i)] = clock64(); g_ta_blk[blockIdx.x * 4 + (i) + 2] = ta_gtime(); } } while (0)
extern "C" void scw_debug_ta_read(long long* out) { cudaMemcpyFromSymbol(out, g_ta_dbg, sizeof(long long) * 8192); }
extern "C" void scw_debug_ta_blk(long long* out) { cudaMemcpyFromSymbol(out, g_ta_blk, sizeof(long long) * 1024); }
#else
#define TA_MARK(slot) do { } while (0)
#define TA_BLK(i) do { } while (0)
#endif

struct TaParams {
    const float2* V[TA_MAX_INST];
    int64_t ldV[TA_MAX_INST];
    int n_inst;
    int64_t R, J;           // R complex rows, J modes (same for every instance of a group)
    const uint8_t* Wt;      // [n_tile][k_block][hi | lo] K-major UMMA images of [W_r | W_i]
    float* part;            // [slot][Fzt][128] fp32 partial tiles
    int N2, Fzt, n_tiles, m_tiles, kblocks, S, stg_stages;
};

// ---- W~ in UMMA image form -----------------------------------------------------------------------
// a-1 mode weights (eq. 7, 30) evaluated in fp64, split to bf16 hi/lo, written as the K-major no-swizzle
// shared-memory image of every (n_tile, k_block) B tile: element (n, kk) at
//   (kk/8)*(N2*16) + (n/8)*128 + (n%8)*16 + (kk%8)*2,  n < Fzt: Re W[j, i], n >= Fzt: Im W[j, i].
struct TwGroup {
    const float2* c[TA_MAX_INST];
    const double2* gamma[TA_MAX_INST];
    const int8_t* dir[TA_MAX_INST];
    const double* z[TA_MAX_INST];
    double inv_lambda[TA_MAX_INST], z_lo[TA_MAX_INST], z_hi[TA_MAX_INST];
};

__global__ void k_tc_weights(int n_inst, int64_t J, int64_t Fz, int Fzt, int n_tiles, int kblocks,
                             const __grid_constant__ TwGroup g_, uint8_t* __restrict__ Wt_all)
{
    const int64_t Jp = (int64_t)kblocks * TA_BK;
    const int64_t per_inst = Jp * n_tiles * Fzt;
    const int64_t gidx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gidx >= per_inst * n_inst) return;
    const int inst = (int)(gidx / per_inst);
    const int64_t idx = gidx - inst * per_inst;
    const float2* __restrict__ c = g_.c[inst];
    const double2* __restrict__ gamma = g_.gamma[inst];
    const int8_t* __restrict__ dir = g_.dir[inst];
    const double* __restrict__ z = g_.z[inst];
    const double inv_lambda = g_.inv_lambda[inst], z_lo = g_.z_lo[inst], z_hi = g_.z_hi[inst];
    uint8_t* Wt = Wt_all + (size_t)inst * n_tiles * kblocks * (size_t)(2 * Fzt) * 256;
    const int64_t i = idx / Jp, j = idx - i * Jp;
    float wr = 0.f, wi = 0.f;
    if (j < J && i < Fz) {
        const double2 g = gamma[j];
        const int d = dir ? (dir[j] > 0 ? 1 : -1) : ((g.y > 0.0 || (g.y == 0.0 && g.x >= 0.0)) ? 1 : -1);
        const double dz = z[i] - (d > 0 ? z_lo : z_hi);
        double t = g.x * dz * inv_lambda;
        t -= rint(t);
        double s, co;
        sincospi(2.0 * t, &s, &co);
        const double a = exp(-6.283185307179586476925 * g.y * dz * inv_lambda);
        double cr = 1.0, ci = 0.0;
        if (c) { cr = (double)c[j].x; ci = (double)c[j].y; }
        wr = (float)(cr * a * co - ci * a * s);
        wi = (float)(cr * a * s + ci * a * co);
    }
    const int N2 = 2 * Fzt;
    const int nt = (int)(i / Fzt), n = (int)(i - (int64_t)nt * Fzt);
    const int kb = (int)(j / TA_BK), kk = (int)(j - (int64_t)kb * TA_BK);
    uint8_t* tile = Wt + ((size_t)nt * kblocks + kb) * (size_t)N2 * 256;
    const size_t off_r = (size_t)(kk >> 3) * (N2 * 16) + (size_t)(n >> 3) * 128 + (n & 7) * 16 + (kk & 7) * 2;
    const int n2 = n + Fzt;
    const size_t off_i = (size_t)(kk >> 3) * (N2 * 16) + (size_t)(n2 >> 3) * 128 + (n2 & 7) * 16 + (kk & 7) * 2;
    const __nv_bfloat16 rh = __float2bfloat16_rn(wr), ih = __float2bfloat16_rn(wi);
    const __nv_bfloat16 rl = __float2bfloat16_rn(wr - __bfloat162float(rh));
    const __nv_bfloat16 il = __float2bfloat16_rn(wi - __bfloat162float(ih));
    const size_t lo = (size_t)N2 * 128;
    *reinterpret_cast<__nv_bfloat16*>(tile + off_r) = rh;
    *reinterpret_cast<__nv_bfloat16*>(tile + off_i) = ih;
    *reinterpret_cast<__nv_bfloat16*>(tile + lo + off_r) = rl;
    *reinterpret_cast<__nv_bfloat16*>(tile + lo + off_i) = il;
}

// ---- main kernel -----------------------------------------------------------------------------------
struct TaPos { int kb, mt, nt, inst; };            // iteration order: instance, n-tile, m-tile, k-block (fastest)

__device__ __forceinline__ TaPos ta_pos(const TaParams& p, int64_t it)
{
    const int64_t tile = it / p.kblocks;
    const int64_t g = tile / p.m_tiles;
    TaPos q;
    q.kb = (int)(it - tile * p.kblocks);
    q.mt = (int)(tile - g * p.m_tiles);
    q.inst = (int)(g / p.n_tiles);
    q.nt = (int)(g - (int64_t)q.inst * p.n_tiles);
    return q;
}
__device__ __forceinline__ void ta_next(const TaParams& p, TaPos& q)
{
    if (++q.kb == p.kblocks) {
        q.kb = 0;
        if (++q.mt == p.m_tiles) {
            q.mt = 0;
            if (++q.nt == p.n_tiles) { q.nt = 0; ++q.inst; }
        }
    }
}

// A V column segment (64 complex rows = 512 B) starts at a 16-byte boundary only when (V/8 + k*ldV) is even;
// otherwise the bulk copy starts 8 bytes early ("shift" = 8).  The shift depends on the parity of k only.
__device__ __forceinline__ uint32_t ta_shift(const float2* V, int64_t ldV, int k_parity)
{
    return (uint32_t)(((reinterpret_cast<uintptr_t>(V) >> 3) + (uint64_t)(k_parity & (int)(ldV & 1))) & 1) * 8u;
}
// Copies move whole 16-byte granules: the window [shift + nvalid*8) is rounded UP (reading one neighbouring
// element of V) unless that would leave the V allocation, in which case it is rounded DOWN and the cut-off
// last row of that column ("tail") is read directly by its converter thread.
__device__ __forceinline__ bool ta_tail_cut(int64_t ldV, int64_t J, int64_t k, int64_t row0, int nvalid, uint32_t sh)
{
    return ((sh + (uint32_t)nvalid * 8u) & 15u) && (k * ldV + row0 + nvalid + 1 > ldV * J);
}

// V-loader warp w copies column segments 8w..8w+7 of the iteration at `q` into a staging slot (lanes 0-7, one
// bulk copy each; a single warp issues only ~1 copy per 80 clk, eight warps together reach ~1 per 16 clk);
// lane 0 posts the warp's byte count on the slot's barrier (one of TA_LOAD_WARPS arrivals).
__device__ __forceinline__ void ta_issue_columns(const TaParams& p, const TaPos q, uint8_t* stg, uint64_t* bar, int w,
                                                 int lane)
{
    const float2* V = p.V[q.inst];
    const int64_t ldV = p.ldV[q.inst];
    const int64_t row0 = (int64_t)q.mt * (TA_BM / 2);
    const int nvalid = (int)min((int64_t)(TA_BM / 2), p.R - row0);
    const int kl = w * 8 + (lane & 7);
    const int64_t k = (int64_t)q.kb * TA_BK + kl;
    const uint32_t sh = ta_shift(V, ldV, lane & 1);
    uint32_t bytes = 0;
    if (lane < 8 && k < p.J) {
        const uint32_t need = sh + (uint32_t)nvalid * 8u;
        bytes = ta_tail_cut(ldV, p.J, k, row0, nvalid, sh) ? (need & ~15u) : ((need + 15u) & ~15u);
    }
    uint32_t total = bytes;
    total += __shfl_xor_sync(0xffffffffu, total, 1);
    total += __shfl_xor_sync(0xffffffffu, total, 2);
    total += __shfl_xor_sync(0xffffffffu, total, 4);
    if (lane == 0) mbar_expect_tx(bar, total);
    __syncwarp();
    if (bytes)
        bulk_g2s(stg + kl * TA_COL_PITCH, reinterpret_cast<const uint8_t*>(V + k * ldV + row0) - sh, bytes, bar);
}

// Converter warp w: TMEM lane quarter q = w & 3 (real rows 32q..32q+31 of the tile), mode half kh = w >> 2
// (modes 32kh..32kh+31 of the stage).  A thread reads its row's 32 fp32 values from the staging slot ([k][row],
// conflict-free 4-byte loads), splits them to bf16 hi/lo pairs and writes them to the A operand block in TMEM
// (lane = row, 32-bit column c holds modes 2c, 2c+1): the tensor core then reads A from TMEM (no shared-memory
// round trip for the converted tile).
__device__ __forceinline__ void ta_convert(const TaParams& p, const uint8_t* stg, uint32_t tmem_a, const TaPos q,
                                           int warp, int lane)
{
    const float2* V = p.V[q.inst];
    const int64_t ldV = p.ldV[q.inst];
    const int64_t row0 = (int64_t)q.mt * (TA_BM / 2);
    const int nvalid = (int)min((int64_t)(TA_BM / 2), p.R - row0);
    const uint32_t sh0 = ta_shift(V, ldV, 0), sh1 = ta_shift(V, ldV, 1);
    const int q4 = warp & 3, kh = warp >> 2;
    const int r = 32 * q4 + lane;                                 // real row in tile: complex row r/2, part r&1
    const uint8_t* src0 = stg + kh * 32 * TA_COL_PITCH + r * 4 + sh0;     // even modes
    const uint8_t* src1 = stg + kh * 32 * TA_COL_PITCH + r * 4 + sh1;     // odd modes
    float v[32];
#pragma unroll
    for (int kk = 0; kk < 32; ++kk) v[kk] = *reinterpret_cast<const float*>(((kk & 1) ? src1 : src0) + kk * TA_COL_PITCH);
    // ragged edges: rows past R and modes past J read as zero (the staging slot holds stale data there)
    const int rc = r >> 1;
    const int klim = (int)min((int64_t)32, p.J - ((int64_t)q.kb * TA_BK + kh * 32));      // warp-uniform
    if (rc >= nvalid || klim < 32) {
#pragma unroll
        for (int kk = 0; kk < 32; ++kk)
            if (rc >= nvalid || kk >= klim) v[kk] = 0.f;
    }
    // the one element a rounded-down copy can cut off: last row of the last column when V has no padding rows
    if (q.kb == p.kblocks - 1 && row0 + nvalid == ldV && rc == nvalid - 1) {
        const int kk = (int)(p.J - 1 - ((int64_t)q.kb * TA_BK + kh * 32));
        if (kk >= 0 && kk < 32 && ta_tail_cut(ldV, p.J, p.J - 1, row0, nvalid, (kk & 1) ? sh1 : sh0)) {
            const float t = __ldg(reinterpret_cast<const float*>(V + (p.J - 1) * ldV + row0 + rc) + (r & 1));
#pragma unroll
            for (int i = 0; i < 32; ++i)
                if (i == kk) v[i] = t;
        }
    }
    uint32_t hi[16], lo[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) split_bf16x2(v[2 * i], v[2 * i + 1], hi[i], lo[i]);
    const uint32_t taddr = tmem_a + ((uint32_t)(32 * q4) << 16) + 16 * kh;
    tmem_st16(taddr, hi);
    tmem_st16(taddr + 32, lo);
    tmem_st_wait();
}

__global__ void __launch_bounds__(TA_THREADS, 1) k_tc_assemble(const __grid_constant__ TaParams p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int mma_stage_bytes = p.N2 * 256;             // W~ tile (hi | lo); the A operand lives in TMEM
    uint8_t* stg_base = smem + (size_t)TA_MMA_STAGES * mma_stage_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(stg_base + (size_t)p.stg_stages * TA_STG_BYTES);
    uint64_t* full_a = bars;                          // converters -> MMA           [TA_MMA_STAGES]
    uint64_t* full_b = full_a + TA_MMA_STAGES;        // W bulk copy -> MMA          [TA_MMA_STAGES]
    uint64_t* empty = full_b + TA_MMA_STAGES;         // MMA commit -> converters, W [TA_MMA_STAGES]
    uint64_t* acc_full = empty + TA_MMA_STAGES;       // MMA commit -> epilogue      [2]
    uint64_t* acc_empty = acc_full + 2;               // epilogue -> MMA             [2]
    uint64_t* stg_full = acc_empty + 2;               // V bulk copies -> converters [stg_stages]
    uint64_t* stg_empty = stg_full + p.stg_stages;    // converters -> V loader      [stg_stages]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(stg_empty + p.stg_stages);

    if (tid == 0) {
        for (int s = 0; s < TA_MMA_STAGES; ++s) {
            mbar_init(&full_a[s], TA_CONV_WARPS * 32);
            mbar_init(&full_b[s], 1);
            mbar_init(&empty[s], 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(&acc_full[b], 1);
            mbar_init(&acc_empty[b], 4);
        }
        for (int s = 0; s < p.stg_stages; ++s) {
            mbar_init(&stg_full[s], TA_LOAD_WARPS);
            mbar_init(&stg_empty[s], TA_CONV_WARPS);
        }
        mbar_fence_init();
    }
    if (warp == TA_MMA_WARP) tmem_alloc(tmem_slot, TA_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    TA_BLK(0);
    const int64_t T = (int64_t)p.n_inst * p.n_tiles * p.m_tiles * p.kblocks;
    const int64_t it0 = (int64_t)blockIdx.x * T / gridDim.x;
    const int64_t it1 = (int64_t)(blockIdx.x + 1) * T / gridDim.x;

    if (warp < TA_CONV_WARPS) {
        // ===== converters: fp32 staging -> bf16 hi/lo UMMA tiles =====
        int sa = 0, ss = 0;
        uint32_t pa = 0, ps = 0;
        TaPos cur = ta_pos(p, it0);
        for (int64_t it = it0; it < it1; ++it) {
            const int dn = (int)(it - it0);
            if (warp == 0) {                       // one warp polls, the other seven sleep on a named barrier
                if (lane == 0) TA_MARK(dn * 16 + 0);
                mbar_wait(&stg_full[ss], ps);
                if (lane == 0) TA_MARK(dn * 16 + 1);
                mbar_wait(&empty[sa], pa ^ 1);
                if (lane == 0) TA_MARK(dn * 16 + 2);
            }
            named_bar_sync(1, TA_CONV_WARPS * 32);
            tc_fence_after();
            if (warp == 0 && lane == 0) TA_MARK(dn * 16 + 3);
            ta_convert(p, stg_base + (size_t)ss * TA_STG_BYTES, tmem_base + TA_A_COL + sa * 64, cur, warp, lane);
            if (warp == 0 && lane == 0) TA_MARK(dn * 16 + 4);
            tc_fence_before();
            mbar_arrive(&full_a[sa]);
            __syncwarp();
            if (lane == 0) mbar_arrive(&stg_empty[ss]);
            if (warp == 0 && lane == 0) TA_MARK(dn * 16 + 5);
            ta_next(p, cur);
            if (++sa == TA_MMA_STAGES) { sa = 0; pa ^= 1; }
            if (++ss == p.stg_stages) { ss = 0; ps ^= 1; }
        }
    } else if (warp < TA_W_LOADER) {
        // ===== V loaders: keep stg_stages x 32 KB of bulk copies in flight =====
        int ss = 0;
        uint32_t ps = 0;
        TaPos q = ta_pos(p, it0);
        for (int64_t it = it0; it < it1; ++it) {
            mbar_wait(&stg_empty[ss], ps ^ 1);
            ta_issue_columns(p, q, stg_base + (size_t)ss * TA_STG_BYTES, &stg_full[ss], warp - TA_V_LOADER, lane);
            ta_next(p, q);
            if (++ss == p.stg_stages) { ss = 0; ps ^= 1; }
        }
    } else if (warp == TA_W_LOADER) {
        // ===== W tile loader (bulk async copy, completes on full_b) =====
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            const uint32_t bytes = (uint32_t)p.N2 * 256;
            for (int64_t it = it0; it < it1; ++it) {
                const int64_t tile = it / p.kblocks;
                const int kb = (int)(it - tile * p.kblocks);
                const int nt = (int)(tile / p.m_tiles);
                mbar_wait(&empty[stage], phase ^ 1);
                mbar_expect_tx(&full_b[stage], bytes);
                bulk_g2s(smem + (size_t)stage * mma_stage_bytes,
                         p.Wt + ((size_t)nt * p.kblocks + kb) * bytes, bytes, &full_b[stage]);
                if (++stage == TA_MMA_STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == TA_MMA_WARP) {
        // ===== MMA issuer: the whole warp runs the loop (warp-uniform descriptors), one elected lane issues =====
        const uint32_t idesc = umma_idesc_bf16(TA_BM, p.N2);
        const uint32_t b_lbo = (uint32_t)p.N2 * 16;
        const uint32_t smem0 = smem_u32(smem);
        int stage = 0, buf = 0;
        uint32_t phase = 0, use0 = 0, use1 = 0;
        int64_t it = it0;
        while (it < it1) {
            const int64_t tile = it / p.kblocks;
            const int64_t seg_end = min(it1, (tile + 1) * p.kblocks);
            const uint32_t use = buf ? use1 : use0;
            mbar_wait(&acc_empty[buf], (use & 1) ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + (uint32_t)(buf * p.N2);
            uint32_t acc = 0;
            for (; it < seg_end; ++it) {
                TA_MARK((int)(it - it0) * 16 + 8);
                mbar_wait(&full_a[stage], phase);
                TA_MARK((int)(it - it0) * 16 + 9);
                mbar_wait(&full_b[stage], phase);
                tc_fence_after();
                TA_MARK((int)(it - it0) * 16 + 10);
                const uint32_t a_hi = tmem_base + TA_A_COL + (uint32_t)stage * 64;     // TMEM columns
                const uint32_t a_lo = a_hi + 32;
                const uint32_t b_hi = smem0 + (uint32_t)stage * (uint32_t)mma_stage_bytes;
                const uint32_t b_lo = b_hi + (uint32_t)p.N2 * 128;
                const uint64_t db_hi0 = umma_desc(b_hi, b_lbo, 128), db_lo0 = umma_desc(b_lo, b_lbo, 128);
                if (elect_one()) {
#pragma unroll
                    for (int s = 0; s < TA_BK / 16; ++s) {
                        const uint64_t kb = (uint64_t)((s * 2 * b_lbo) >> 4);
                        umma_bf16_ts(d_tmem, a_lo + 8 * s, db_hi0 + kb, idesc, acc);
                        acc = 1;
                        umma_bf16_ts(d_tmem, a_hi + 8 * s, db_lo0 + kb, idesc, 1);
                        umma_bf16_ts(d_tmem, a_hi + 8 * s, db_hi0 + kb, idesc, 1);
                    }
                    umma_commit(&empty[stage]);
                }
                __syncwarp();
                acc = 1;
                TA_MARK((int)(it - it0) * 16 + 11);
                if (++stage == TA_MMA_STAGES) { stage = 0; phase ^= 1; }
            }
            if (elect_one()) umma_commit(&acc_full[buf]);
            __syncwarp();
            if (buf) ++use1; else ++use0;
            buf ^= 1;
        }
    } else {
        // ===== epilogue: TMEM -> registers -> lane-pair combine -> partial tile =====
        const int q = warp & 3;                                   // TMEM lane quarter this warp may access
        int buf = 0, seg = 0;
        uint32_t use0 = 0, use1 = 0;
        int64_t it = it0;
        while (it < it1) {
            const int64_t tile = it / p.kblocks;
            const int64_t seg_end = min(it1, (tile + 1) * p.kblocks);
            if (q == 0) mbar_wait(&acc_full[buf], (buf ? use1 : use0) & 1);
            named_bar_sync(10, 128);
            tc_fence_after();
            float* out = p.part + ((size_t)blockIdx.x * p.S + seg) * ((size_t)p.Fzt * TA_BM) + 32 * q + lane;
            const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(buf * p.N2);
            for (int i0 = 0; i0 < p.Fzt; i0 += 8) {
                float a[8], b[8];
                tmem_ld8(taddr + i0, a);
                tmem_ld8(taddr + p.Fzt + i0, b);
                tmem_ld_wait();
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const float recv = __shfl_xor_sync(0xffffffffu, b[e], 1);
                    // even lane: Re = D[2r,i] - D[2r+1,Fzt+i];  odd lane: Im = D[2r+1,i] + D[2r,Fzt+i]
                    out[(size_t)(i0 + e) * TA_BM] = (lane & 1) ? a[e] + recv : a[e] - recv;
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&acc_empty[buf]);
            if (buf) ++use1; else ++use0;
            buf ^= 1;
            ++seg;
            it = seg_end;
        }
    }
    tc_fence_before();
    __syncthreads();
    TA_BLK(1);
    if (warp == TA_MMA_WARP) tmem_dealloc(tmem_base, TA_TMEM_COLS);
}

// Sum the segments of every tile in CTA order: P[mt*64 + r, nt*Fzt + n] = sum_seg part[seg][n][2r..2r+1].
__global__ void k_tc_reduce(int64_t R, int64_t Fz, int Fzt, int n_tiles, int m_tiles, int kblocks, int64_t T, int G, int S,
                            const float* __restrict__ part, float2* __restrict__ P_all, int64_t ldP, int64_t inst_stride)
{
    const int tile = blockIdx.x;                                 // global tile id: (inst, n_tile, m_tile)
    const int n = blockIdx.y * blockDim.y + threadIdx.y;
    const int r = threadIdx.x;                                   // complex row in tile, 0..63
    const int gnt = tile / m_tiles, mt = tile - gnt * m_tiles;
    const int inst = gnt / n_tiles, nt = gnt - inst * n_tiles;
    float2* __restrict__ P = P_all + (int64_t)inst * inst_stride;
    const int64_t row = (int64_t)mt * 64 + r, col = (int64_t)nt * Fzt + n;
    if (n >= Fzt || row >= R || col >= Fz) return;
    const int64_t a = (int64_t)tile * kblocks, b = a + kblocks;
    const int c_first = (int)(((a + 1) * G + T - 1) / T) - 1;
    const int c_last = (int)((b * G + T - 1) / T) - 1;
    float2 acc = make_float2(0.f, 0.f);
    for (int c = c_first; c <= c_last; ++c) {
        const int64_t start = (int64_t)c * T / G;
        const int seg = tile - (int)(start / kblocks);
        const float2 v = *reinterpret_cast<const float2*>(part + ((size_t)c * S + seg) * ((size_t)Fzt * TA_BM) +
                                                          (size_t)n * TA_BM + 2 * r);
        acc.x += v.x;
        acc.y += v.y;
    }
    P[row + col * ldP] = acc;
}

// ---- host side -------------------------------------------------------------------------------------
struct TaPlan {
    int Fzt, N2, n_tiles, m_tiles, kblocks, G, S, stg_stages;
    int64_t T;
    size_t wt_bytes, part_bytes, smem_bytes;      // wt_bytes: W~ images of ONE instance
};

static TaPlan ta_plan(int64_t R, int64_t J, int64_t Fz, int n_inst, int sm_count)
{
    TaPlan pl;
    int64_t fzt = (Fz + 7) / 8 * 8;
    if (fzt > 64) fzt = 64;
    pl.Fzt = (int)fzt;
    pl.N2 = 2 * pl.Fzt;
    pl.n_tiles = (int)((Fz + pl.Fzt - 1) / pl.Fzt);
    pl.m_tiles = (int)((2 * R + TA_BM - 1) / TA_BM);
    pl.kblocks = (int)((J + TA_BK - 1) / TA_BK);
    pl.T = (int64_t)n_inst * pl.n_tiles * pl.m_tiles * pl.kblocks;
    pl.G = (int)(pl.T < sm_count ? pl.T : sm_count);
    pl.S = 1;
    for (int c = 0; c < pl.G; ++c) {
        const int64_t s = (int64_t)c * pl.T / pl.G, e = (int64_t)(c + 1) * pl.T / pl.G;
        if (e > s) {
            const int span = (int)((e - 1) / pl.kblocks - s / pl.kblocks) + 1;
            if (span > pl.S) pl.S = span;
        }
    }
    const int mma_bytes = TA_MMA_STAGES * (pl.N2 * 256);
    pl.stg_stages = (TA_SMEM_LIMIT - 256 - mma_bytes) / TA_STG_BYTES;
    if (pl.stg_stages > 5) pl.stg_stages = 5;
    pl.smem_bytes = (size_t)mma_bytes + (size_t)pl.stg_stages * TA_STG_BYTES + 256;
    pl.wt_bytes = (size_t)pl.n_tiles * pl.kblocks * pl.N2 * 256;
    pl.part_bytes = align_up((size_t)pl.G * pl.S * pl.Fzt * TA_BM * sizeof(float));
    return pl;
}

bool tc_assemble_supported(int dtype, int64_t R, int64_t J, int64_t Fz)
{
    return dtype == SCW_C64 && R >= 1 && J >= 1 && Fz >= 1;
}

int tc_assemble_max_group() { return TA_MAX_INST; }

size_t tc_assemble_scratch(int64_t R, int64_t J, int64_t Fz, int n_inst, int sm_count)
{
    const TaPlan pl = ta_plan(R, J, Fz, n_inst, sm_count);
    return align_up(pl.wt_bytes * n_inst) + pl.part_bytes;
}

// A group of n_inst <= TA_MAX_INST instances with the same U, Vn, J and Fz in three launches:
// weights (a-1), P = V W over the concatenated iteration space (a-2), segment reduce.
// Instance i writes P_all + i * inst_stride (column-major [ldP x Fz]).
void launch_tc_assemble_group(scw_ctx* ctx, int n_inst, const scw_layer* inst, int64_t Fz, const double* const* z,
                              void* P_all, int64_t ldP, int64_t inst_stride, void* scratch)
{
    const scw_layer& L0 = inst[0];
    const int64_t R = 3LL * L0.U * L0.Vn;
    const TaPlan pl = ta_plan(R, L0.J, Fz, n_inst, ctx->sm_count);
    uint8_t* Wt = static_cast<uint8_t*>(scratch);
    float* part = reinterpret_cast<float*>(Wt + align_up(pl.wt_bytes * n_inst));
    TwGroup g;
    TaParams p;
    for (int i = 0; i < n_inst; ++i) {
        g.c[i] = (const float2*)inst[i].c;
        g.gamma[i] = (const double2*)inst[i].gamma;
        g.dir[i] = inst[i].dir;
        g.z[i] = z[i];
        g.inv_lambda[i] = 1.0 / inst[i].lambda;
        g.z_lo[i] = inst[i].z_lo;
        g.z_hi[i] = inst[i].z_hi;
        p.V[i] = (const float2*)inst[i].V;
        p.ldV[i] = inst[i].ldV;
    }
    {
        KernelScope ks(ctx, KC_WEIGHTS);
        const int64_t n = (int64_t)pl.kblocks * TA_BK * pl.n_tiles * pl.Fzt * n_inst;
        k_tc_weights<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(n_inst, L0.J, Fz, pl.Fzt, pl.n_tiles,
                                                                           pl.kblocks, g, Wt);
    }
    p.n_inst = n_inst;
    p.R = R;
    p.J = L0.J;
    p.Wt = Wt;
    p.part = part;
    p.N2 = pl.N2;
    p.Fzt = pl.Fzt;
    p.n_tiles = pl.n_tiles;
    p.m_tiles = pl.m_tiles;
    p.kblocks = pl.kblocks;
    p.S = pl.S;
    p.stg_stages = pl.stg_stages;
    {
        KernelScope ks(ctx, KC_ASSEMBLE_TC);
        cudaFuncSetAttribute(k_tc_assemble, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes);
        k_tc_assemble<<<pl.G, TA_THREADS, pl.smem_bytes, ctx->stream>>>(p);
    }
    {
        KernelScope ks(ctx, KC_REDUCE);
        dim3 block(64, 4);
        dim3 grid((unsigned)(n_inst * pl.n_tiles * pl.m_tiles), (unsigned)((pl.Fzt + 3) / 4));
        k_tc_reduce<<<grid, block, 0, ctx->stream>>>(R, Fz, pl.Fzt, pl.n_tiles, pl.m_tiles, pl.kblocks, pl.T, pl.G, pl.S,
                                                     part, (float2*)P_all, ldP, inst_stride);
    }
}

void launch_tc_assemble(scw_ctx* ctx, const scw_layer* L, int64_t Fz, const double* z, void* P, int64_t ldP,
                        void* scratch)
{
    launch_tc_assemble_group(ctx, 1, L, Fz, &z, P, ldP, 0, scratch);
}

}  // namespace scw
