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
// Work decomposition ("stream-K"): the iteration space (instance, n_tile, m_tile, k_block) is cut into
// equal contiguous spans, one per persistent CTA (one CTA per SM); every (CTA, tile) segment writes an
// fp32 partial tile, k_tc_reduce sums the segments of each tile in a fixed order (deterministic).
//
// A tile is 128 complex rows (two 128-lane M blocks) x 32 modes per pipeline stage.  V reaches shared
// memory through TMA: two tensor maps per instance describe the even and the odd columns of V (column
// stride 2*ldV*8 bytes is a multiple of 16 for any ldV; for odd ldV the odd-column map starts one element
// early with a 130-row box so that every box starts on a 16-byte boundary), so one elected thread issues two
// 16 KB box copies per stage --
// 1 KB contiguous per column, rows past R and columns past J arrive as zeros.
// Warp roles (768 threads): warps 0-15 (two groups of 8 on alternate stages) read their real row of the
// staged fp32 tile, split it to bf16 hi/lo and write the A operand straight into TMEM (tcgen05.st); warp 16 =
// TMA producer for V; warp 17 fetches the pre-formatted W tiles with bulk copies; warp 18 issues tcgen05.mma
// (A from TMEM, B from shared memory); warps 20-23 drain the accumulators (tcgen05.ld), combine lanes with
// one shuffle per element and store the partial tile.
#include <cuda.h>

#include "scw_internal.h"
#include "scw_tc_common.cuh"

namespace scw {

using namespace tc;

constexpr int TA_ROWS = 128;               // complex rows per tile (= 256 real rows = 2 M blocks of 128 lanes)
constexpr int TA_BK = 32;                  // modes per pipeline stage: even modes in staging columns 0-15, odd in 16-31
constexpr int TA_CONV_WARPS = 8;           // converter warp w of a group owns real rows 32w..32w+31 of the tile
constexpr int TA_CONV_GROUPS = 2;          // group g converts the CTA's iterations n = g, g+2, ... (two stages in flight)
constexpr int TA_V_LOADER = 16, TA_W_LOADER = 17, TA_MMA_WARP = 18, TA_EPI_WARP0 = 20;
constexpr int TA_THREADS = 24 * 32;
constexpr int TA_A_COL = 256;              // TMEM: A operand, per MMA stage and M block 16 columns hi + 16 columns lo
constexpr int TA_STG_ODD = TA_ROWS * 8 * 16;          // fp32 staging slot: [16 even columns][128 rows] then the odd-column box
constexpr int TA_STG_BYTES = TA_STG_ODD + 16 * (TA_ROWS + 2) * 8;   // odd-column box: up to 130 rows (odd ldV, see ta_make_map)
constexpr int TA_MMA_STAGES = 3;
constexpr int TA_TMEM_COLS = 512;
constexpr int TA_SMEM_LIMIT = 226 * 1024;
constexpr int TA_MAX_STG = 5;

constexpr int TA_MAX_INST = 64;            // instances (layers x wavelengths) per grouped launch


struct TaParams {
    CUtensorMap tmap[TA_MAX_INST][2];   // [0]: even columns of V, [1]: odd columns; box = 128 rows x 16 columns of 8 bytes
    int xoff1[TA_MAX_INST];             // 1 when ldV is odd: odd-column box has 130 rows and starts one element early
    int n_inst;
    const uint8_t* Wt;      // [inst][n_tile][k_block][hi | lo] K-major UMMA images of [W_r | W_i]
    float* part;            // [slot][Fzt][256] fp32 partial tiles
    int* seg_count;         // [tile] number of stream-K segments of the tile (written by the tile's first CTA)
    int* seg_slot;          // [tile][max_segs] slot of every segment, in CTA order
    int N2, Fzt, n_tiles, m_tiles, kblocks, S, stg_stages, nbuf, max_segs;
};

// Mode index of staging column kk (0..31) of k-block kb: even modes first, then odd modes.
__host__ __device__ __forceinline__ int64_t ta_mode(int kb, int kk)
{
    return (int64_t)kb * TA_BK + (kk < 16 ? 2 * kk : 2 * (kk - 16) + 1);
}

// ---- W~ in UMMA image form -----------------------------------------------------------------------
// a-1 mode weights (eq. 7, 30): phase reduced in fp64 (turns), sincospi / exp in fp32 (the result is split to
// bf16 hi + lo, 2^-17 relative, so fp32 transcendentals lose nothing), written as the K-major no-swizzle
// shared-memory image of every (n_tile, k_block) B tile: element (n, kk) at
//   (kk/8)*(N2*16) + (n/8)*128 + (n%8)*16 + (kk%8)*2,  n < Fzt: Re W[j, i], n >= Fzt: Im W[j, i],  j = ta_mode(kb, kk).
// One thread produces two consecutive kk (4 bytes of a 16-byte core-matrix row), for the Re and the Im row, hi and lo.
struct TwGroup {
    const float2* c[TA_MAX_INST];
    const double2* gamma[TA_MAX_INST];
    const int8_t* dir[TA_MAX_INST];
    const double* z[TA_MAX_INST];
    double inv_lambda[TA_MAX_INST], z_lo[TA_MAX_INST], z_hi[TA_MAX_INST];
};

__global__ void __launch_bounds__(256) k_tc_weights(int n_inst, int64_t J, int64_t Fz, int Fzt, int n_tiles, int kblocks,
                                                    const __grid_constant__ TwGroup g_, uint8_t* __restrict__ Wt_all)
{
    // block = one (inst, n_tile, k_block) tile; thread item = (k chunk c4, plane n, mode pair e2), e2 fastest: the four
    // lanes of a pair group fill one 16-byte core-matrix row, a warp writes 128 contiguous bytes per store
    const int kb = blockIdx.x, nt = blockIdx.y, inst = blockIdx.z;
    const int64_t tile_id = ((int64_t)inst * n_tiles + nt) * kblocks + kb;
    const float2* __restrict__ c = g_.c[inst];
    const double2* __restrict__ gamma = g_.gamma[inst];
    const int8_t* __restrict__ dir = g_.dir[inst];
    const double inv_lambda = g_.inv_lambda[inst], z_lo = g_.z_lo[inst], z_hi = g_.z_hi[inst];
    const int N2 = 2 * Fzt;
    uint8_t* tile = Wt_all + (size_t)tile_id * (size_t)N2 * 128;
    for (int rem = threadIdx.x; rem < 16 * Fzt; rem += blockDim.x) {
    const int e2 = rem & 3, cn = rem >> 2;
    const int c4 = cn / Fzt, n = cn - c4 * Fzt;                        // k chunk (8 modes), plane within the n tile
    const int64_t i = (int64_t)nt * Fzt + n;
    const double zi = i < Fz ? g_.z[inst][i] : 0.0;
    float wr[2], wi[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const int64_t j = ta_mode(kb, 8 * c4 + 2 * e2 + e);
        wr[e] = 0.f;
        wi[e] = 0.f;
        if (j < J && i < Fz) {
            const double2 g = gamma[j];
            const int d = dir ? (dir[j] > 0 ? 1 : -1) : ((g.y > 0.0 || (g.y == 0.0 && g.x >= 0.0)) ? 1 : -1);
            const double dz = (zi - (d > 0 ? z_lo : z_hi)) * inv_lambda;
            // phase in turns, reduced in fp64 by the magic-constant trick: the low word of t + 1.5*2^20 is
            // frac(t) * 2^32 (two's complement: an angle in [-pi, pi) after scaling), then the MUFU sin / cos / ex2
            // (abs. error ~5e-7, below the 2^-17 of the bf16 hi/lo split that follows)
            // (the product is reduced with rint first, so a thick layer with |gamma dz / lambda| >= 2^19 turns is fine)
            const double tt = g.x * dz;
            const int ph = __double2loint((tt - rint(tt)) + 1572864.0);
            const float ang = __int2float_rn(ph) * 1.4629180792671596e-9f;           // 2 pi / 2^32
            const float s = __sinf(ang), co = __cosf(ang);
            const float a = exp2f((float)(-9.0647202836543876194 * g.y * dz));        // exp(-2 pi x) = 2^(-2 pi log2(e) x)
            float cr = 1.f, ci = 0.f;
            if (c) { cr = c[j].x; ci = c[j].y; }
            const float ar = a * co, ai = a * s;
            wr[e] = cr * ar - ci * ai;
            wi[e] = cr * ai + ci * ar;
        }
    }
    uint32_t rh, rl, ih, il;
    split_bf16x2(wr[0], wr[1], rh, rl);
    split_bf16x2(wi[0], wi[1], ih, il);
    const int n2 = n + Fzt;
    const size_t off_r = (size_t)c4 * (N2 * 16) + (size_t)(n >> 3) * 128 + (n & 7) * 16 + e2 * 4;
    const size_t off_i = (size_t)c4 * (N2 * 16) + (size_t)(n2 >> 3) * 128 + (n2 & 7) * 16 + e2 * 4;
    const size_t lo = (size_t)N2 * 64;
    *reinterpret_cast<uint32_t*>(tile + off_r) = rh;
    *reinterpret_cast<uint32_t*>(tile + off_i) = ih;
    *reinterpret_cast<uint32_t*>(tile + lo + off_r) = rl;
    *reinterpret_cast<uint32_t*>(tile + lo + off_i) = il;
    }
}

// ---- main kernel -----------------------------------------------------------------------------------
struct TaPos { int kb, mt, g, nt, inst; };   // iteration order: g = (instance, n-tile), m-tile, k-block (fastest)

__device__ __forceinline__ TaPos ta_pos(const TaParams& p, int64_t it)
{
    const int64_t tile = it / p.kblocks;
    TaPos q;
    q.kb = (int)(it - tile * p.kblocks);
    q.g = (int)(tile / p.m_tiles);
    q.mt = (int)(tile - (int64_t)q.g * p.m_tiles);
    q.inst = q.g / p.n_tiles;
    q.nt = q.g - q.inst * p.n_tiles;
    return q;
}
__device__ __forceinline__ void ta_next(const TaParams& p, TaPos& q)
{
    if (++q.kb == p.kblocks) {
        q.kb = 0;
        if (++q.mt == p.m_tiles) {
            q.mt = 0;
            ++q.g;
            if (++q.nt == p.n_tiles) { q.nt = 0; ++q.inst; }
        }
    }
}

__global__ void __launch_bounds__(TA_THREADS, 1) k_tc_assemble(const __grid_constant__ TaParams p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int w_stage_bytes = p.N2 * 128;               // W~ tile (hi | lo) of one stage; the A operand lives in TMEM
    uint8_t* stg_base = smem;                           // fp32 staging ring (TMA destination, 32 KB slots)
    uint8_t* w_base = smem + (size_t)p.stg_stages * TA_STG_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(w_base + (size_t)TA_MMA_STAGES * w_stage_bytes);
    uint64_t* full_a = bars;                          // converters -> MMA           [TA_MMA_STAGES]
    uint64_t* full_b = full_a + TA_MMA_STAGES;        // W bulk copy -> MMA          [TA_MMA_STAGES]
    uint64_t* empty = full_b + TA_MMA_STAGES;         // MMA commit -> converters, W [TA_MMA_STAGES]
    uint64_t* acc_full = empty + TA_MMA_STAGES;       // MMA commit -> epilogue      [2]
    uint64_t* acc_empty = acc_full + 2;               // epilogue -> MMA             [2]
    uint64_t* stg_full = acc_empty + 2;               // TMA -> converters           [stg_stages]
    uint64_t* stg_empty = stg_full + TA_MAX_STG;      // converters -> TMA producer  [stg_stages]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(stg_empty + TA_MAX_STG);

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
            mbar_init(&stg_full[s], 1);
            mbar_init(&stg_empty[s], TA_CONV_WARPS);
        }
        mbar_fence_init();
    }
    if (warp == TA_MMA_WARP) tmem_alloc(tmem_slot, TA_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int64_t T = (int64_t)p.n_inst * p.n_tiles * p.m_tiles * p.kblocks;
    const int64_t it0 = (int64_t)blockIdx.x * T / gridDim.x;
    const int64_t it1 = (int64_t)(blockIdx.x + 1) * T / gridDim.x;

    if (warp < TA_CONV_WARPS * TA_CONV_GROUPS) {
        // ===== converters: staged fp32 -> bf16 hi/lo A operand in TMEM =====
        // Two groups of 8 warps take alternate iterations, so that the shared-memory loads, the split arithmetic and
        // the TMEM stores of two stages overlap.  Thread = real row r = 32*w + lane of the tile (w = warp within the
        // group; complex row r/2, part r&1): M block w>>2, TMEM lane quarter w&3.  It reads its 32 fp32 values of the
        // stage ([column][row] layout: conflict-free 4-byte loads), splits them and writes 16 + 16 columns (bf16
        // pairs: column c holds staging columns 2c, 2c+1).
        const int grp = warp >> 3, w = warp & 7;
        int sa = 0, ss = 0;
        uint32_t pa = 0, ps = 0;
        TaPos cur = ta_pos(p, it0);
        auto advance = [&]() {
            ta_next(p, cur);
            if (++sa == TA_MMA_STAGES) { sa = 0; pa ^= 1; }
            if (++ss == p.stg_stages) { ss = 0; ps ^= 1; }
        };
        if (grp == 1) advance();
        const uint32_t a_lane = tmem_base + TA_A_COL + (uint32_t)((w >> 2) * 32) + ((uint32_t)(32 * (w & 3)) << 16);
        for (int64_t it = it0 + grp; it < it1; it += TA_CONV_GROUPS) {
            if (w == 0) {                          // one warp polls, the other seven sleep on a named barrier
                mbar_wait(&stg_full[ss], ps);
                mbar_wait(&empty[sa], pa ^ 1);
            }
            named_bar_sync(1 + grp, TA_CONV_WARPS * 32);
            tc_fence_after();
            const uint8_t* src = stg_base + (size_t)ss * TA_STG_BYTES + (32 * w + lane) * 4;
            float v[32];
#pragma unroll
            for (int kk = 0; kk < 16; ++kk) v[kk] = *reinterpret_cast<const float*>(src + kk * (TA_ROWS * 8));
            if (p.xoff1[cur.inst]) {               // odd ldV: odd-column box is 130 rows, data starts one element in
#pragma unroll
                for (int kk = 0; kk < 16; ++kk)
                    v[16 + kk] = *reinterpret_cast<const float*>(src + TA_STG_ODD + 8 + kk * ((TA_ROWS + 2) * 8));
            } else {
#pragma unroll
                for (int kk = 0; kk < 16; ++kk)
                    v[16 + kk] = *reinterpret_cast<const float*>(src + TA_STG_ODD + kk * (TA_ROWS * 8));
            }
            uint32_t hi[16], lo[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) split_bf16x2(v[2 * i], v[2 * i + 1], hi[i], lo[i]);
            const uint32_t taddr = a_lane + (uint32_t)sa * 64;
            tmem_st16(taddr, hi);
            tmem_st16(taddr + 16, lo);
            __syncwarp();
            if (lane == 0) mbar_arrive(&stg_empty[ss]);        // staging slot is in registers now
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(&full_a[sa]);
            advance();
            advance();
        }
    } else if (warp == TA_V_LOADER) {
        // ===== TMA producer: two 128-row x 16-column boxes (even / odd modes) per stage =====
        if (lane == 0) {
            int ss = 0;
            uint32_t ps = 0;
            TaPos q = ta_pos(p, it0);
            for (int64_t it = it0; it < it1; ++it) {
                const int inst = q.inst;
                uint8_t* dst = stg_base + (size_t)ss * TA_STG_BYTES;
                mbar_wait(&stg_empty[ss], ps ^ 1);
                mbar_expect_tx(&stg_full[ss], TA_STG_ODD + 16 * (TA_ROWS + 2 * p.xoff1[inst]) * 8);
                tma_load_2d(dst, &p.tmap[inst][0], q.mt * TA_ROWS, q.kb * 16, &stg_full[ss]);
                tma_load_2d(dst + TA_STG_ODD, &p.tmap[inst][1], q.mt * TA_ROWS, q.kb * 16, &stg_full[ss]);
                ta_next(p, q);
                if (++ss == p.stg_stages) { ss = 0; ps ^= 1; }
            }
        }
    } else if (warp == TA_W_LOADER) {
        // ===== W tile loader (bulk async copy, completes on full_b) =====
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            const uint32_t bytes = (uint32_t)w_stage_bytes;
            TaPos q = ta_pos(p, it0);
            for (int64_t it = it0; it < it1; ++it) {
                mbar_wait(&empty[stage], phase ^ 1);
                mbar_expect_tx(&full_b[stage], bytes);
                bulk_g2s(w_base + (size_t)stage * w_stage_bytes, p.Wt + ((size_t)q.g * p.kblocks + q.kb) * bytes, bytes,
                         &full_b[stage]);
                ta_next(p, q);
                if (++stage == TA_MMA_STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == TA_MMA_WARP) {
        // ===== MMA issuer: the whole warp runs the loop (warp-uniform descriptors), one elected lane issues =====
        const uint32_t idesc = umma_idesc_bf16(128, p.N2);
        const uint32_t b_lbo = (uint32_t)p.N2 * 16;
        const uint32_t w0 = smem_u32(w_base);
        int stage = 0, buf = 0;
        uint32_t phase = 0, use0 = 0, use1 = 0;
        int64_t it = it0;
        while (it < it1) {
            const int64_t tile = it / p.kblocks;
            const int64_t seg_end = min(it1, (tile + 1) * p.kblocks);
            const uint32_t use = buf ? use1 : use0;
            mbar_wait(&acc_empty[buf], (use & 1) ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + (uint32_t)(buf * 2 * p.N2);
            uint32_t acc = 0;
            for (; it < seg_end; ++it) {
                mbar_wait(&full_a[stage], phase);
                mbar_wait(&full_b[stage], phase);
                tc_fence_after();
                const uint32_t a0 = tmem_base + TA_A_COL + (uint32_t)stage * 64;       // TMEM columns: block b at +32b, lo at +16
                const uint32_t b_hi = w0 + (uint32_t)stage * (uint32_t)w_stage_bytes;
                const uint32_t b_lo = b_hi + (uint32_t)p.N2 * 64;
                const uint64_t db_hi0 = umma_desc(b_hi, b_lbo, 128), db_lo0 = umma_desc(b_lo, b_lbo, 128);
                if (elect_one()) {
#pragma unroll
                    for (int b = 0; b < 2; ++b) {
                        const uint32_t d = d_tmem + (uint32_t)(b * p.N2);
                        const uint32_t a_hi = a0 + 32 * b, a_lo = a_hi + 16;
#pragma unroll
                        for (int s = 0; s < TA_BK / 16; ++s) {
                            const uint64_t kofs = (uint64_t)((s * 2 * b_lbo) >> 4);
                            umma_bf16_ts(d, a_lo + 8 * s, db_hi0 + kofs, idesc, s == 0 ? acc : 1u);
                            umma_bf16_ts(d, a_hi + 8 * s, db_lo0 + kofs, idesc, 1);
                            umma_bf16_ts(d, a_hi + 8 * s, db_hi0 + kofs, idesc, 1);
                        }
                    }
                    umma_commit(&empty[stage]);
                }
                __syncwarp();
                acc = 1;
                if (++stage == TA_MMA_STAGES) { stage = 0; phase ^= 1; }
            }
            if (elect_one()) umma_commit(&acc_full[buf]);
            __syncwarp();
            if (buf) ++use1; else ++use0;
            if (p.nbuf == 2) buf ^= 1;
        }
    } else if (warp >= TA_EPI_WARP0) {
        // ===== epilogue: TMEM -> registers -> lane-pair combine -> partial tile [plane][256 real rows] =====
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
            if (q == 0 && lane == 0) {
                // segment table: the CTAs whose spans meet this tile are c_first..c_last, this one is number c - c_first
                const int64_t a = tile * p.kblocks, b = a + p.kblocks;
                const int c_first = (int)(((a + 1) * gridDim.x + T - 1) / T) - 1;
                p.seg_slot[tile * p.max_segs + ((int)blockIdx.x - c_first)] = (int)blockIdx.x * p.S + seg;
                if ((int)blockIdx.x == c_first) p.seg_count[tile] = (int)((b * gridDim.x + T - 1) / T) - c_first;
            }
            float* out = p.part + ((size_t)blockIdx.x * p.S + seg) * ((size_t)p.Fzt * 2 * TA_ROWS) + 32 * q + lane;
#pragma unroll 1
            for (int b = 0; b < 2; ++b) {
                const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(buf * 2 * p.N2 + b * p.N2);
                int i0 = 0;
                for (; i0 + 16 <= p.Fzt; i0 += 16) {              // 16 planes per TMEM round trip
                    float a[16], bb[16];
                    tmem_ld16(taddr + i0, a);
                    tmem_ld16(taddr + p.Fzt + i0, bb);
                    tmem_ld_wait();
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        const float recv = __shfl_xor_sync(0xffffffffu, bb[e], 1);
                        // even lane: Re = D[2r,i] - D[2r+1,Fzt+i];  odd lane: Im = D[2r+1,i] + D[2r,Fzt+i]
                        out[(size_t)(i0 + e) * (2 * TA_ROWS) + b * 128] = (lane & 1) ? a[e] + recv : a[e] - recv;
                    }
                }
                for (; i0 < p.Fzt; i0 += 8) {                     // Fzt is a multiple of 8
                    float a[8], bb[8];
                    tmem_ld8(taddr + i0, a);
                    tmem_ld8(taddr + p.Fzt + i0, bb);
                    tmem_ld_wait();
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const float recv = __shfl_xor_sync(0xffffffffu, bb[e], 1);
                        out[(size_t)(i0 + e) * (2 * TA_ROWS) + b * 128] = (lane & 1) ? a[e] + recv : a[e] - recv;
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&acc_empty[buf]);
            if (buf) ++use1; else ++use0;
            if (p.nbuf == 2) buf ^= 1;
            ++seg;
            it = seg_end;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == TA_MMA_WARP) tmem_dealloc(tmem_base, TA_TMEM_COLS);
}

// Sum the segments of every tile in CTA order: P[mt*128 + r, nt*Fzt + n] = sum_seg part[seg][n][2r..2r+1].
__global__ void k_tc_reduce(int64_t R, int64_t Fz, int Fzt, int n_tiles, int m_tiles, int max_segs,
                            const int* __restrict__ seg_count, const int* __restrict__ seg_slot,
                            const float* __restrict__ part, float2* __restrict__ P_all, int64_t ldP, int64_t inst_stride)
{
    const int tile = blockIdx.x;                                 // global tile id: (inst, n_tile, m_tile)
    const int n = blockIdx.y * blockDim.y + threadIdx.y;
    const int r = threadIdx.x;                                   // complex row in tile, 0..127
    const int gnt = tile / m_tiles, mt = tile - gnt * m_tiles;
    const int inst = gnt / n_tiles, nt = gnt - inst * n_tiles;
    float2* __restrict__ P = P_all + (int64_t)inst * inst_stride;
    const int64_t row = (int64_t)mt * TA_ROWS + r, col = (int64_t)nt * Fzt + n;
    if (n >= Fzt || row >= R || col >= Fz) return;
    const int count = seg_count[tile];
    const int* __restrict__ slots = seg_slot + (size_t)tile * max_segs;
    float2 acc = make_float2(0.f, 0.f);
    for (int i = 0; i < count; ++i) {
        const float2 v = *reinterpret_cast<const float2*>(part + (size_t)slots[i] * ((size_t)Fzt * 2 * TA_ROWS) +
                                                          (size_t)n * (2 * TA_ROWS) + 2 * r);
        acc.x += v.x;
        acc.y += v.y;
    }
    P[row + col * ldP] = acc;
}

// ---- host side -------------------------------------------------------------------------------------
struct TaPlan {
    int Fzt, N2, n_tiles, m_tiles, kblocks, G, S, stg_stages, nbuf, max_segs;
    int64_t T;
    size_t wt_bytes, part_bytes, seg_bytes, smem_bytes;      // wt_bytes: W~ images of ONE instance
};

static TaPlan ta_plan(int64_t R, int64_t J, int64_t Fz, int n_inst, int sm_count)
{
    TaPlan pl;
    int64_t fzt = (Fz + 7) / 8 * 8;
    if (fzt > 64) fzt = 64;
    pl.Fzt = (int)fzt;
    pl.N2 = 2 * pl.Fzt;
    pl.nbuf = pl.N2 <= 64 ? 2 : 1;                // TMEM: 256 accumulator columns, 2 M blocks of N2 each per buffer
    pl.n_tiles = (int)((Fz + pl.Fzt - 1) / pl.Fzt);
    pl.m_tiles = (int)((R + TA_ROWS - 1) / TA_ROWS);
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
    const int w_bytes = TA_MMA_STAGES * (pl.N2 * 128);
    pl.stg_stages = (TA_SMEM_LIMIT - 256 - w_bytes) / TA_STG_BYTES;
    if (pl.stg_stages > TA_MAX_STG) pl.stg_stages = TA_MAX_STG;
    pl.smem_bytes = (size_t)w_bytes + (size_t)pl.stg_stages * TA_STG_BYTES + 256;
    pl.wt_bytes = (size_t)pl.n_tiles * pl.kblocks * pl.N2 * 128;
    pl.part_bytes = align_up((size_t)pl.G * pl.S * pl.Fzt * 2 * TA_ROWS * sizeof(float));
    // a CTA span holds at least T/G iterations, so at most (kblocks-1)/(T/G) + 2 spans meet one tile
    pl.max_segs = (int)((pl.kblocks - 1) / (pl.T / pl.G) + 2);
    pl.seg_bytes = align_up((size_t)n_inst * pl.n_tiles * pl.m_tiles * (1 + pl.max_segs) * sizeof(int));
    return pl;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libscw does not link libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// Tensor map over every second column of V starting at column `first` (0 or 1): 8-byte elements,
// dim0 = rows (contiguous), dim1 = columns at stride 2*ldV*8 bytes; box 128 x 16; out-of-range reads give 0.
// L2 promotion 64 B: the 1 KB column pieces start at arbitrary 8-byte offsets, wider promotion re-fetches the
// boundary lines shared with the vertically adjacent tile (measured: 256 B -> 64 B = 112 -> 104 us at config 1).
// For odd ldV the odd columns start 8 bytes off a 16-byte boundary: their map starts one element earlier (the last
// element of the column before) and its box is 130 rows, so that every box still starts on a 16-byte boundary
// (TMA faults otherwise); row r of the tile then sits at box row r + 1 (xoff = 1).
static bool ta_make_map(CUtensorMap* map, const void* V, int64_t ldV, int64_t R, int64_t J, int first, int* xoff)
{
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const int off = (first == 1 && (ldV & 1)) ? 1 : 0;
    const char* base = static_cast<const char*>(V) + (size_t)first * ldV * 8 - (size_t)off * 8;
    int64_t ncols = first == 0 ? (J + 1) / 2 : J / 2;
    if (ncols < 1) { ncols = 1; base = static_cast<const char*>(V); }      // J == 1: never addressed with valid data
    const cuuint64_t dims[2] = {(cuuint64_t)(R + off), (cuuint64_t)ncols};
    const cuuint64_t strides[1] = {(cuuint64_t)(2 * ldV * 8)};
    const cuuint32_t box[2] = {(cuuint32_t)(TA_ROWS + 2 * off), 16};
    const cuuint32_t estr[2] = {1, 1};
    if (xoff) *xoff = off;
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, const_cast<char*>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// TMA needs a 16-byte aligned base and strides below 2^40 bytes; J >= 2 keeps the odd-column map non-empty.
bool tc_assemble_supported(int dtype, int64_t R, int64_t J, int64_t Fz, const void* V, int64_t ldV)
{
    return dtype == SCW_C64 && R >= 1 && J >= 2 && Fz >= 1 && (reinterpret_cast<uintptr_t>(V) & 15) == 0 &&
           2 * ldV * 8 < ((int64_t)1 << 40) && R + 1 < ((int64_t)1 << 32) && (Fz + 63) / 64 <= 65535;
}

int tc_assemble_max_group() { return TA_MAX_INST; }

size_t tc_assemble_scratch(int64_t R, int64_t J, int64_t Fz, int n_inst, int sm_count)
{
    const TaPlan pl = ta_plan(R, J, Fz, n_inst, sm_count);
    return align_up(pl.wt_bytes * n_inst) + pl.part_bytes + pl.seg_bytes;
}

// weights (a-1) + the stream-K assembly kernel (a-2) of a group; the partial tiles end up in `part`.
static bool ta_run(scw_ctx* ctx, int n_inst, const scw_layer* inst, int64_t Fz, const double* const* z, void* scratch,
                   TaPlan& pl, float*& part, int*& seg_count, int*& seg_slot)
{
    const scw_layer& L0 = inst[0];
    const int64_t R = 3LL * L0.U * L0.Vn;
    pl = ta_plan(R, L0.J, Fz, n_inst, ctx->sm_count);
    uint8_t* Wt = static_cast<uint8_t*>(scratch);
    part = reinterpret_cast<float*>(Wt + align_up(pl.wt_bytes * n_inst));
    seg_count = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(part) + pl.part_bytes);
    seg_slot = seg_count + (size_t)n_inst * pl.n_tiles * pl.m_tiles;
    TwGroup g;
    static thread_local TaParams p;                 // 17 KB of kernel parameters: kept off the stack
    bool maps_ok = true;
    for (int i = 0; i < n_inst; ++i) {
        g.c[i] = (const float2*)inst[i].c;
        g.gamma[i] = (const double2*)inst[i].gamma;
        g.dir[i] = inst[i].dir;
        g.z[i] = z[i];
        g.inv_lambda[i] = 1.0 / inst[i].lambda;
        g.z_lo[i] = inst[i].z_lo;
        g.z_hi[i] = inst[i].z_hi;
        maps_ok = maps_ok && ta_make_map(&p.tmap[i][0], inst[i].V, inst[i].ldV, R, L0.J, 0, nullptr) &&
                  ta_make_map(&p.tmap[i][1], inst[i].V, inst[i].ldV, R, L0.J, 1, &p.xoff1[i]);
    }
    if (!maps_ok) {                                 // reported by the entry point's check_launch
        ctx->tc_error = true;
        return false;
    }
    {
        KernelScope ks(ctx, KC_WEIGHTS);
        const dim3 grid((unsigned)pl.kblocks, (unsigned)pl.n_tiles, (unsigned)n_inst);
        k_tc_weights<<<grid, 256, 0, ctx->stream>>>(n_inst, L0.J, Fz, pl.Fzt, pl.n_tiles, pl.kblocks, g, Wt);
    }
    p.n_inst = n_inst;
    p.Wt = Wt;
    p.part = part;
    p.seg_count = seg_count;
    p.seg_slot = seg_slot;
    p.max_segs = pl.max_segs;
    p.N2 = pl.N2;
    p.Fzt = pl.Fzt;
    p.n_tiles = pl.n_tiles;
    p.m_tiles = pl.m_tiles;
    p.kblocks = pl.kblocks;
    p.S = pl.S;
    p.stg_stages = pl.stg_stages;
    p.nbuf = pl.nbuf;
    {
        KernelScope ks(ctx, KC_ASSEMBLE_TC);
        cudaFuncSetAttribute(k_tc_assemble, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes);
        k_tc_assemble<<<pl.G, TA_THREADS, pl.smem_bytes, ctx->stream>>>(p);
    }
    return true;
}

void launch_tc_assemble_group_partials(scw_ctx* ctx, int n_inst, const scw_layer* inst, int64_t Fz, const double* const* z,
                                       void* scratch, TcPartials* out)
{
    TaPlan pl;
    float* part = nullptr;
    int *seg_count = nullptr, *seg_slot = nullptr;
    out->part = nullptr;
    if (!ta_run(ctx, n_inst, inst, Fz, z, scratch, pl, part, seg_count, seg_slot)) return;
    out->part = part;
    out->seg_count = seg_count;
    out->seg_slot = seg_slot;
    out->max_segs = pl.max_segs;
    out->Fzt = pl.Fzt;
    out->n_tiles = pl.n_tiles;
    out->m_tiles = pl.m_tiles;
    out->rows_per_tile = TA_ROWS;
}

// A group of n_inst <= TA_MAX_INST instances with the same U, Vn, J and Fz in three launches:
// weights (a-1), P = V W over the concatenated iteration space (a-2), segment reduce.
// Instance i writes P_all + i * inst_stride (column-major [ldP x Fz]).
void launch_tc_assemble_group(scw_ctx* ctx, int n_inst, const scw_layer* inst, int64_t Fz, const double* const* z,
                              void* P_all, int64_t ldP, int64_t inst_stride, void* scratch)
{
    TaPlan pl;
    float* part = nullptr;
    int *seg_count = nullptr, *seg_slot = nullptr;
    if (!ta_run(ctx, n_inst, inst, Fz, z, scratch, pl, part, seg_count, seg_slot)) return;
    const int64_t R = 3LL * inst[0].U * inst[0].Vn;
    KernelScope ks(ctx, KC_REDUCE);
    dim3 block(TA_ROWS, 2);
    dim3 grid((unsigned)(n_inst * pl.n_tiles * pl.m_tiles), (unsigned)((pl.Fzt + 1) / 2));
    k_tc_reduce<<<grid, block, 0, ctx->stream>>>(R, Fz, pl.Fzt, pl.n_tiles, pl.m_tiles, pl.max_segs, seg_count, seg_slot,
                                                 part, (float2*)P_all, ldP, inst_stride);
}

void launch_tc_assemble(scw_ctx* ctx, const scw_layer* L, int64_t Fz, const double* z, void* P, int64_t ldP,
                        void* scratch)
{
    launch_tc_assemble_group(ctx, 1, L, Fz, &z, P, ldP, 0, scratch);
}

}  // namespace scw
