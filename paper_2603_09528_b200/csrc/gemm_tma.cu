// gemm_tma.cu — the eigenbasis transforms (steps 2.1, 2.2, 2.4, 2.5) as a persistent,
// warp-specialised FP64 tensor-path GEMM for sm_100a.
//
//   * FP64 has no tcgen05 path: the FP64 tensor unit of sm_100 is reached through mma.sync m8n8k4 (SASS DMMA.8x8x4).
//   * one CTA per SM, static round-robin over 128x128 output tiles; 16 consumer warps (32x32 warp tiles, 64 FP64
//     accumulators per lane, setmaxnreg 112) + a producer warpgroup (setmaxnreg 24) whose elected lane feeds a STAGES-deep ring of k-slabs (16 k each)
//     by TMA (SASS UTMALDG); full/empty mbarriers per slot — no CTA-wide barrier anywhere in the main loop, so
//     warps drift apart by up to a ring's worth of slabs and the epilogue of one tile overlaps the loads of the next.
//   * operands land in shared memory in the TMA 128-byte swizzle; the rows of every 8-row group and the columns of
//     every 16-column group are assigned to MMA lanes through fixed permutations (rho, nu below) that make every
//     64-bit fragment load bank-conflict free without padding.
//
// Row-major C[b] (M x N) = A[b] (M x K, k contiguous) * B[b] (K x N, n contiguous).  Any M and K, any even N ("the
// framework supports non-uniform grids in any direction", PAPER.md:187 — any N_x, N_y): ragged edge tiles are loaded
// with TMA's out-of-bounds zero fill (a zero row of A or column of B contributes nothing), warps whose 32x32 sub-tile
// lies wholly outside skip their DMMAs, and the epilogue stores are predicated.
#include <cuda.h>

#include "devonce.hpp"
#include "kernels.cuh"
#include "ptx.cuh"
#include "tmap.hpp"

namespace tpt {

namespace {

constexpr int BM = 128, BN = 128, BK = 16;
constexpr int CONSUMER_WARPS = 16;
constexpr int THREADS = (CONSUMER_WARPS + 4) * 32;   // + one producer warpgroup (register budgets are per warpgroup)
constexpr int A_BYTES = BM * BK * 8;          // 16 KB: 128 rows of 128 B
constexpr int B_BYTES = BK * BN * 8;          // 16 KB: 8 sub-tiles [16 k][16 n] of 2 KB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
constexpr int STAGES = 6;
constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 2 * STAGES * 8;

struct TmaGemmParams {
    double *C;
    int64_t ldc, strideC;
    int64_t ldg;         // stride between 16-column groups of C (16 = plain row-major)
    int M, N;            // extents of C (edge tiles: predicated stores)
    int KT;              // ceil(K / 16)
    int tiles_n;         // ceil(N / 128)
    int tiles_mn;        // ceil(M / 128) * ceil(N / 128)
    int ntiles;          // tiles_mn * batch
    int b_split;         // N % 16 != 0: mapB is the plain 3-D tensor [batch][K][N], one load per 16-column group
    int a_batch_rows;    // rows of the A tensor per batch (0: shared by all batches)
    int b_batch_rows;    // rows of the B tensor per batch (0: shared)
    // sharded solve: rows of C scattered to their owners' memory (GemmArgs::peerC); row m belongs to rank
    // ((m/16 + 1) * npeers - 1) / units, the inverse of the unit split [units*q/npeers, units*(q+1)/npeers)
    int npeers, units;
    double *peerC[MAX_PEERS];
};

// EDGE = false: M, N multiples of 128 and K of 16 — no predicate, no skipped warp, plain stride-grid tile walk (the
// round-1 kernel, instruction for instruction: the headline configs).  EDGE = true: everything described above.
template <bool EDGE>
__global__ void __launch_bounds__(THREADS, 1)
gemm_tma_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                const TmaGemmParams p) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)STAGES * STAGE_BYTES);
    uint64_t *empty = full + STAGES;

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        ptx::tma_prefetch_desc(&mapA);
        ptx::tma_prefetch_desc(&mapB);
        for (int s = 0; s < STAGES; ++s) {
            ptx::mbar_init(&full[s], 1);
            ptx::mbar_init(&empty[s], CONSUMER_WARPS);
        }
        ptx::fence_mbar_init();
    }
    ptx::pdl_launch_dependents();
    __syncthreads();
    ptx::pdl_wait();              // the operands are the previous kernel's output

    const int KT = p.KT;
    if (warp >= CONSUMER_WARPS) {
        // ---------------- producer warpgroup: one elected lane --------------------------------------
        ptx::setmaxnreg_dec<24>();
        if (warp == CONSUMER_WARPS && lane == 0) {
            int slot = 0;
            uint32_t phase = 0;
            for (int round = 0, base = 0; base < p.ntiles; ++round, base += gridDim.x) {
                const int tile = base + (EDGE ? (int)((blockIdx.x + round) % gridDim.x) : (int)blockIdx.x);
                if (tile >= p.ntiles) continue;
                const int b = tile / p.tiles_mn;
                const int mn = tile - b * p.tiles_mn;
                const int mt = mn / p.tiles_n, nt = mn - mt * p.tiles_n;
                const int a_row = b * p.a_batch_rows + mt * BM;
                const int b_sel = p.b_batch_rows ? b : 0;
                for (int kt = 0; kt < KT; ++kt) {
                    ptx::mbar_wait(&empty[slot], phase ^ 1);
                    unsigned char *st = smem + (size_t)slot * STAGE_BYTES;
                    ptx::mbar_arrive_expect_tx(&full[slot], STAGE_BYTES);
                    ptx::tma_load_2d(st, &mapA, kt * BK, a_row, &full[slot]);
                    if (!EDGE || !p.b_split) {
                        ptx::tma_load_4d(st + A_BYTES, &mapB, 0, kt * BK, nt * (BN / 16), b_sel, &full[slot]);
                    } else {     // same shared-memory image, built from eight boxes clipped at column N
#pragma unroll
                        for (int q = 0; q < BN / 16; ++q)
                            ptx::tma_load_3d(st + A_BYTES + q * 2048, &mapB, nt * BN + q * 16, kt * BK, b_sel, &full[slot]);
                    }
                    if (++slot == STAGES) { slot = 0; phase ^= 1; }
                }
            }
        }
        return;
    }

    // ---------------- consumers ---------------------------------------------------------------------
    ptx::setmaxnreg_inc<112>();   // 640 x 96 registers at launch = 128 x 24 + 512 x 112 (the pool is the CTA's own)
    const int g = lane >> 2, t = lane & 3;
    // Warp w runs on SM sub-partition w % 4.  The 4 x 4 grid of 32 x 32 warp tiles is handed out as a Latin square: every
    // sub-partition holds one warp of each row block AND of each column block, so on an edge tile (rows or columns past
    // M / N skipped) the remaining DMMAs still spread evenly over the four FP64 tensor pipes.
    const int wm0 = (warp >> 2) * 32, wn0 = (EDGE ? (((warp & 3) + (warp >> 2)) & 3) : (warp & 3)) * 32;
    const int rho = ((g & 3) << 1) | (g >> 2);                 // MMA row g  <-> tile row 8i + rho
    // A fragment (row 8i + rho, k = 4kk + t):  byte = row*128 + (((k>>1) ^ rho) << 4) + (k&1)*8
    uint32_t a_off[4];
    {
        const uint32_t c = (uint32_t)((t >> 1) ^ rho) << 4;
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) a_off[kk] = (uint32_t)(wm0 + rho) * 128u + (c ^ (uint32_t)(kk * 32)) + (t & 1) * 8u;
    }
    // B fragment (k = 4kk + t, column nu(g, tile) of 16-column group sub):
    //   nu = (g&1) | ((g>>2)&1)<<1 | tile<<2 | ((g>>1)&1)<<3 ;  byte = sub*2048 + k*128 + (((nu>>1) ^ (k&7)) << 4) + (nu&1)*8
    uint32_t b_off[2][2];                                      // [tile][kk & 1]
    {
        const uint32_t nb = (uint32_t)(((g >> 2) & 1) | (((g >> 1) & 1) << 2));
        const uint32_t c = nb ^ (uint32_t)t;
#pragma unroll
        for (int tile = 0; tile < 2; ++tile)
#pragma unroll
            for (int kp = 0; kp < 2; ++kp)
                b_off[tile][kp] = (uint32_t)(wn0 / 16) * 2048u + (uint32_t)t * 128u +
                                  ((c ^ (uint32_t)((tile << 1) | (kp << 2))) << 4) + (g & 1) * 8u;
    }
    const uint32_t smem_base = ptx::smem_u32(smem);

    // A slot is handed back to the producer one slab late: the arrive for slab q is issued after the wait for slab
    // q+1, i.e. behind (in issue order) every DMMA of slab q — whose operand scoreboards guarantee that all of
    // slab q's LDS have returned.  Arriving straight after *issuing* the last LDS is not enough: with 16 warps
    // queueing shared-memory loads the read itself can still be pending when an L2-hit TMA refill lands.
    int slot = 0, prev_slot = -1;
    uint32_t phase = 0;
    // Static schedule: round r hands tiles [r grid, (r+1) grid) to the CTAs rotated by r — with a plain stride-grid walk a
    // CTA would meet the same (mt, nt) every round whenever grid is a multiple of tiles_mn, i.e. some CTAs only cheap edge
    // tiles and others only full ones.
    for (int round = 0, base = 0; base < p.ntiles; ++round, base += gridDim.x) {
        const int tile = base + (EDGE ? (int)((blockIdx.x + round) % gridDim.x) : (int)blockIdx.x);
        if (tile >= p.ntiles) continue;
        double acc[4][4][2];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        const int b = tile / p.tiles_mn;
        const int mn = tile - b * p.tiles_mn;
        const int mt = mn / p.tiles_n, nt = mn - mt * p.tiles_n;
        // edge tiles: a warp whose sub-tile lies wholly past M or N only keeps the ring's bookkeeping going
        const bool inside = !EDGE || (mt * BM + wm0 < p.M && nt * BN + wn0 < p.N);

        for (int kt = 0; kt < KT; ++kt) {
            ptx::mbar_wait(&full[slot], phase);
            if (prev_slot >= 0) {
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(&empty[prev_slot]);
            }
            const uint32_t sa = smem_base + (uint32_t)slot * STAGE_BYTES;
            const uint32_t sb = sa + A_BYTES;
            if (inside) {
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
                double af[4], bf[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) af[i] = ptx::lds_f64(sa + a_off[kk] + i * 1024);
#pragma unroll
                for (int j = 0; j < 4; ++j) bf[j] = ptx::lds_f64(sb + b_off[j & 1][kk & 1] + (j >> 1) * 2048 + kk * 512);
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) ptx::dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            }
            }
            prev_slot = slot;
            if (++slot == STAGES) { slot = 0; phase ^= 1; }
        }
        // epilogue: lane holds rows 8i + rho, columns nu(2t), nu(2t)+1 of each MMA tile -> 16-byte stores
        if (!inside) continue;
        const int row0 = mt * BM + wm0 + rho;
        const int cin = ((t >> 1) << 1) + ((t & 1) << 3);          // first of my two columns inside a 16-column group
        const int col0 = nt * BN + wn0 + cin;
        const int64_t off = (int64_t)b * p.strideC + (int64_t)(nt * (BN / 16) + wn0 / 16) * p.ldg + cin;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int row = row0 + 8 * i;
            if (EDGE && row >= p.M) break;
            // sharded solve: the owner of mode row `row` receives it straight from this epilogue (16-byte stores to
            // peer-mapped memory travel over NVLink while the next tile's DMMAs run) — no pack kernel, no collective
            double *base = p.npeers ? p.peerC[(((row >> 4) + 1) * p.npeers - 1) / p.units] : p.C;
            double *Cw = base + off + (int64_t)row * p.ldc;
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (!EDGE || col0 + (j >> 1) * 16 + (j & 1) * 4 < p.N)   // N is even: a column pair is inside or outside as a whole
                    *reinterpret_cast<double2 *>(Cw + (int64_t)(j >> 1) * p.ldg + (j & 1) * 4) = make_double2(acc[i][j][0], acc[i][j][1]);
        }
    }
}

bool aligned16(const void *q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; }

}  // namespace

bool gemm_tma_supported(const GemmArgs &g) {
    if (g.M < 1 || g.N < 2 || g.N % 2 || g.K < 1 || g.batch < 1) return false;
    if (g.lda % 2 || g.ldb % 2 || g.ldc % 2 || g.strideC % 2) return false;
    // the blocked layouts address whole 16-column groups; the peer scatter owns rows in 16-row units
    if ((g.ldgB > 16 || g.ldgC > 16 || g.npeers) && g.N % 16) return false;
    if (g.npeers && g.M % 16) return false;
    if (!aligned16(g.A) || !aligned16(g.B) || !aligned16(g.C)) return false;
    if (g.npeers < 0 || g.npeers > MAX_PEERS) return false;
    for (int q = 0; q < g.npeers; ++q)
        if (!g.peerC[q] || !aligned16(g.peerC[q])) return false;
    // batches are folded into the row dimension of the operand tensors: a batched operand must be densely stacked
    if (g.batch > 1) {
        // a batched A is one tall tensor: its edge tiles would run into the next batch
        if (g.strideA != 0 && (g.strideA != (int64_t)g.M * g.lda || g.M % BM)) return false;
        if (g.strideB != 0 && g.strideB % 2) return false;
    }
    if (g.ldgB % 2 || g.ldgC % 2) return false;
    const int64_t tiles = (int64_t)((g.M + BM - 1) / BM) * ((g.N + BN - 1) / BN) * g.batch;
    return tiles < (int64_t)1 << 30;
}

cudaError_t gemm_tma_configure() {
    // setmaxnreg.inc<112> in the consumers can only be granted from the CTA's own launch allocation:
    // THREADS x numRegs >= 128 x 24 + 512 x 112, i.e. 96 registers per thread at launch (what ptxas gives under
    // __launch_bounds__(640, 1) today).  A toolchain that allocated fewer would hang the kernel: refuse instead.
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, gemm_tma_kernel<false>);
    if (e != cudaSuccess) return e;
    if (fa.numRegs * THREADS < 128 * 24 + CONSUMER_WARPS * 32 * 112) return cudaErrorLaunchOutOfResources;
    e = cudaFuncGetAttributes(&fa, gemm_tma_kernel<true>);
    if (e != cudaSuccess) return e;
    if (fa.numRegs * THREADS < 128 * 24 + CONSUMER_WARPS * 32 * 112) return cudaErrorLaunchOutOfResources;
    e = cudaFuncSetAttribute(gemm_tma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(gemm_tma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES);
}

cudaError_t launch_gemm_tma(const GemmArgs &g, int sms, cudaStream_t stream) {
    if (!gemm_tma_supported(g)) return cudaErrorInvalidValue;
    const bool a_batched = g.batch > 1 && g.strideA != 0;
    const bool b_batched = g.batch > 1 && g.strideB != 0;
    CUtensorMap mapA, mapB;
    {
        const uint64_t dims[2] = {(uint64_t)g.K, (uint64_t)g.M * (a_batched ? g.batch : 1)};
        const uint64_t strides[1] = {(uint64_t)g.lda * 8};
        const uint32_t box[2] = {BK, BM};
        if (!make_f64_map(&mapA, g.A, 2, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B)) return cudaErrorUnknown;
    }
    const bool b_split = g.N % 16 != 0;
    if (b_split) {
        // plain [batch][K][N]: a box is one 16 k x 16 n sub-tile, clipped (zero-filled) at column N
        const uint64_t dims[3] = {(uint64_t)g.N, (uint64_t)g.K, (uint64_t)(b_batched ? g.batch : 1)};
        const uint64_t strides[2] = {(uint64_t)g.ldb * 8, (uint64_t)(b_batched ? g.strideB : (int64_t)g.K * g.ldb) * 8};
        const uint32_t box[3] = {16, BK, 1};
        if (!make_f64_map(&mapB, g.B, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B)) return cudaErrorUnknown;
    } else {
        // B viewed as [batch][N/16 groups][K rows][16 columns]: one box = 8 sub-tiles of 16 k x 16 n (128-byte rows)
        const uint64_t ldg = g.ldgB ? (uint64_t)g.ldgB : 16;
        const uint64_t dims[4] = {16, (uint64_t)g.K, (uint64_t)g.N / 16, (uint64_t)(b_batched ? g.batch : 1)};
        const uint64_t strides[3] = {(uint64_t)g.ldb * 8, ldg * 8, (uint64_t)(b_batched ? g.strideB : (int64_t)g.K * g.ldb) * 8};
        const uint32_t box[4] = {16, BK, BN / 16, 1};
        if (!make_f64_map(&mapB, g.B, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B)) return cudaErrorUnknown;
    }
    TmaGemmParams p;
    p.C = g.C;
    p.ldc = g.ldc;
    p.strideC = g.strideC;
    p.ldg = g.ldgC ? g.ldgC : 16;
    p.M = g.M;
    p.N = g.N;
    p.KT = (g.K + BK - 1) / BK;
    p.tiles_n = (g.N + BN - 1) / BN;
    p.tiles_mn = ((g.M + BM - 1) / BM) * p.tiles_n;
    p.ntiles = p.tiles_mn * g.batch;
    p.b_split = b_split ? 1 : 0;
    p.a_batch_rows = a_batched ? g.M : 0;
    p.b_batch_rows = b_batched ? g.K : 0;
    p.npeers = g.npeers;
    p.units = g.M / 16 > 0 ? g.M / 16 : 1;
    for (int q = 0; q < MAX_PEERS; ++q) p.peerC[q] = q < g.npeers ? g.peerC[q] : nullptr;
    const int grid = p.ntiles < sms ? p.ntiles : sms;
    if (g.M % BM == 0 && g.N % BN == 0 && g.K % BK == 0) return launch_pdl(gemm_tma_kernel<false>, dim3(grid), dim3(THREADS), SMEM_BYTES, stream, mapA, mapB, p);
    return launch_pdl(gemm_tma_kernel<true>, dim3(grid), dim3(THREADS), SMEM_BYTES, stream, mapA, mapB, p);
}

}  // namespace tpt
