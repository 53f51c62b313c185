// kernels.cuh — launch wrappers of the sm_100a kernels (definitions in kernels.cu).
#pragma once

#include <cuda_runtime.h>

#include <cstdint>
#include <vector>

namespace tpt {

// Row-major batched GEMM  C[b] = A[b] * B[b],  A: M x K (lda), B: K x N (ldb), C: M x N (ldc),
// batch strides in elements (0 = operand shared by all batches).
constexpr int MAX_PEERS = 8;   // ranks of a sharded plan: one NVLink domain of 8 GPUs

struct GemmArgs {
    const double *A;
    const double *B;
    double *C;
    int M, N, K;
    int64_t lda, ldb, ldc;
    int64_t strideA, strideB, strideC;
    int batch;
    // Column-group strides (elements) of B and C: column n lives at (n / 16) * ldg + n % 16 within its row.
    // 0 or 16 = plain row-major.  Anything else is the tile-blocked mode-space layout of the y transforms (below);
    // only the TMA kernel (variant 2) takes it.
    int64_t ldgB = 0, ldgC = 0;
    // Sharded solve (sharded.cu): the rows of C are owned by `npeers` ranks in blocks of 16-row units
    // (rank q owns units [units*q/npeers, units*(q+1)/npeers), units = M/16); row m is then written through peerC[q]
    // instead of C — a pointer into rank q's memory (peer-mapped over NVLink), with the owner's row offset and this
    // rank's batch offset already folded in.  npeers == 0: plain single-destination C.  TMA kernel only.
    int npeers = 0;
    double *peerC[MAX_PEERS] = {};
};

// Tile-blocked layout of the mode-space field between steps 2.2 and 2.4 (the z sweep's input and output):
//   element (i, m, k) at  ((m * (nx/16) + i/16) * nz + k) * 16 + i % 16
// i.e. the nz rows of every 16-column Thomas tile are contiguous (nz * 128 bytes), so the sweep reads and writes whole
// DRAM pages instead of one 128-byte line per page (natural layout: rows nx*ny*8 bytes apart; measured 4.6 vs 6.1 TB/s
// for the bare tile traffic).  Written by the forward-y GEMM epilogue, read back by the inverse-y GEMM's B tensor map.
inline bool blocked_layout_supported(int nx, int ny, int nz) { return nx % 16 == 0 && ny >= 1 && nz >= 1; }

// variant 0: generic FP64-FMA tile kernel, any shape.  variant 1: DMMA pipelined kernel when the
// shape allows (falls back to the generic kernel otherwise).  Returns the launch's cudaError_t.
cudaError_t launch_gemm(const GemmArgs &g, int variant, cudaStream_t stream);
bool gemm_dmma_supported(const GemmArgs &g);
cudaError_t gemm_configure();   // one-time cudaFuncSetAttribute for the dynamic-smem kernels

// variant 2 (gemm_tma.cu): persistent warp-specialised DMMA kernel fed by TMA through an mbarrier ring.
// Any M, K and even N (edge tiles through TMA's out-of-bounds zero fill and predicated stores), even leading dimensions,
// 16-byte aligned bases, batched operands densely stacked; the blocked layouts need N % 16 == 0.  sms = SM count.
bool gemm_tma_supported(const GemmArgs &g);
cudaError_t gemm_tma_configure();
cudaError_t launch_gemm_tma(const GemmArgs &g, int sms, cudaStream_t stream);

// z sweep (step 2.3): in place on x (nx*ny*nz), cprime = field-sized scratch.
// Solves (T_z + (lamx[i] + lamy[j] + shift0) I) x = rhs for each column; on a singular plan the
// column (0,0) gets "last unknown = 0".
// b0_null: diagonal entry of row 0 for the null column (= bz[0] except in the cyclic sweep, see launch_cyclic_*).
cudaError_t launch_thomas(double *x, double *cprime, const double *az, const double *bz, const double *cz,
                          const double *lamx, const double *lamy, int nx, int ny, int nz, double shift0,
                          int singular, double b0_null, cudaStream_t stream);

// Periodic z (A19): Sherman-Morrison correction around the tridiagonal sweep (kernels.cu).
// Natural layout, cols = nx * ny.  rhs: u = (g, 0, .., 0, cn) in every column; rden from the swept q; correct: per solve.
cudaError_t launch_cyclic_rhs(double *u, size_t cols, int nz, double g, double cn, cudaStream_t stream);
cudaError_t launch_cyclic_rden(const double *q, double *rden, size_t cols, int nz, double r, int singular, cudaStream_t stream);
cudaError_t launch_cyclic_correct(double *x, const double *q, const double *rden, size_t cols, int nz, double r, cudaStream_t stream);

// Same solve with the z-columns resident on chip (thomas_onchip.cu): 16 B/pt of HBM traffic, no scratch field.
// Reads the right-hand sides from `in` and writes the solution to `x` (in == x: in place).
// tab: device copy of the tables thomas_onchip_tables() builds (16 * (nz + THOMAS_TABLE_PAD) doubles: regular and null-column
// table for each of the two partitions — blocked / natural launch shape — in the kernel's order: groups of 4 segments, row-interleaved).
// sms = SM count.
constexpr int THOMAS_TABLE_PAD = 160;   // >= the rows by which S*M can exceed nz in any launch shape
bool thomas_onchip_supported(int nx, int ny, int nz);
// b_null: diagonal of the null column's table when it differs from b (cyclic sweep: unmodified corners); nullptr = b.
void thomas_onchip_tables(int nz, const double *a, const double *b, const double *c, std::vector<double> &out,
                          const double *b_null = nullptr);
bool thomas_onchip_geometry(int nz, bool blocked_any, bool sharded, int out[12]);   // launch shape of an nz (thomas_onchip.cu)
// wz: the nz cell widths of the z direction — on a singular plan the kernel itself removes the dz-weighted mean of the
// null column (0,0) before the tile leaves the chip (A7): no separate gauge launch.
cudaError_t launch_thomas_onchip(const double *in, double *x, const double *tab, const double *lamx, const double *lamy, const double *wz,
                                 int nx, int ny, int nz, double shift0, int singular, bool blocked, bool blocked_shape, int sms,
                                 cudaStream_t stream);

// Sharded solve (sharded.cu): the sweep over the `rows` y-modes this rank owns (field `in`: tile-blocked, rows * nx
// columns, full nz), the solution rows [k0[r], k0[r+1]) of every tile stored into rank r's z-slab buffer slab[r]
// (tile-blocked over ALL total_cols = nx*ny columns with that rank's nz_r rows; peer-mapped memory).
struct ThomasPeers {
    int npeers = 0;
    int k0[MAX_PEERS + 1] = {};       // slab boundaries; k0[npeers] = nz; even (see launch_thomas_onchip_sharded)
    double *slab[MAX_PEERS] = {};
    size_t total_cols = 0;            // nx * ny
    int group0 = 0;                   // (first owned row) * nx / 16
};
cudaError_t launch_thomas_onchip_sharded(const double *in, const ThomasPeers &peers, const double *tab, const double *lamx,
                                         const double *lamy_owned, const double *wz, int nx, int rows, int nz, double shift0,
                                         int singular, int sms, cudaStream_t stream);

// The whole solve in one cluster launch for grids that fit on chip (fused_small.cu): steps 2.1-2.5 + gauge, GEMM
// transforms only.  work: a field-sized scratch in global memory (the plan's workspace); rhs == out allowed.
struct FusedSmallArgs {
    const double *rhs;
    double *out, *work;
    const double *xfwd, *xinv, *yfwd, *yinv;                  // pre-scaled matrices of the plan (plan.hpp); unused ones may be null
    const double *az, *bz, *cz, *wz, *lamx, *lamy;
    int nx, ny, nz, dirs, singular;
    double shift0;
};
bool fused_small_supported(int nx, int ny, int nz);
cudaError_t launch_fused_small(const FusedSmallArgs &a, cudaStream_t stream);
// The same launch with `work` replaced by a static device array of STATIC_SCRATCH_POINTS doubles (a.work is ignored): no
// allocation on the call path.  cudaErrorInvalidValue beyond that size.  Calls that overlap on one GPU race on the array.
constexpr size_t STATIC_SCRATCH_POINTS = 16384;   // = TPT_STATIC_SCRATCH_POINTS (tpt.h)
cudaError_t launch_fused_small_static(const FusedSmallArgs &a, cudaStream_t stream);

// Null-mode gauge: subtract the dz-weighted mean of column (0,0) (zero volume-weighted mean); `stride` = distance
// between consecutive z levels of that column (nx*ny in the natural layout, 16 in the tile-blocked one).
cudaError_t launch_gauge(double *x, const double *wz, size_t stride, int nz, cudaStream_t stream);

// Staggered-grid operators of the pressure projection, Eq. 2c-2e (projection.cu).  Device vectors of the plan:
// rw* = 1 / cell width (n entries), gf* = 1 / centre spacing at every face (n + 1 entries; boundary faces: one cell
// width, periodic: the wrap spacing).  bc as in tpt.h.
struct ProjGeom {
    int nx, ny, nz;
    int bc[3];
    const double *rwx, *rwy, *rwz, *gfx, *gfy, *gfz;
};
// out = scale * D(u, v, w)
cudaError_t launch_divergence(const double *u, const double *v, const double *w, const ProjGeom &g, double scale,
                              double *out, cudaStream_t stream);
// u -= c G phi (all three face arrays); if p: p += phi - alpha L_I phi, L_I = the directions in `dirs` (z always)
cudaError_t launch_correct(const double *phi, double *u, double *v, double *w, double *p, const ProjGeom &g, double c,
                           double alpha, int dirs, cudaStream_t stream);

// Fast transforms of a uniform direction (fft.cu): the same Eq. 10 / 12 as the GEMM kernels, in the
// field's natural layout.  dir 0: along x for ny*planes rows; dir 1: along y for `planes` z-planes (nx % 16 == 0).
// s0 / s1: scale of the special slots (norm^2 N) / of the others — forward: applied to the outputs, inverse: to the inputs.
struct FftArgs {
    const double *in;
    double *out;
    const double *tables;   // device copy of fft_tables(N)
    int dir, inverse, bc;
    int nx, ny, planes;
    double s0, s1;
    // y only: the mode-space side (output of the forward, input of the inverse transform) is tile-blocked; in / out
    // then point at the FIELD on that side, nz = field depth, k0 = z index of the first plane of this launch
    int blocked = 0, nz = 0, k0 = 0;
    // y only: transform just the columns [x0, x0 + ncols) of every plane (ncols = 0: all nx).  The natural-layout side keeps
    // the full field addressing (row length nx); a blocked side is then a SLAB buffer of its own, ncols columns wide
    // (element (i, m, k) at ((m (ncols/16) + (i - x0)/16) nz + k) 16 + i mod 16) — the L2-resident slab pipeline of api.cu.
    int x0 = 0, ncols = 0;
    // Sharded solve (sharded.cu), forward y with a blocked output only: mode row m belongs to rank ((m/16 + 1) npeers - 1) / units
    // (units = ny / 16) and is stored through peer_out[q] instead of `out` — a pointer into rank q's mode buffer with the
    // owner's row offset folded in; nz / k0 then describe that buffer (full depth, this rank's first plane).
    int npeers = 0;
    double *peer_out[MAX_PEERS] = {};
};
bool fft_supported(int n);                                   // 2^m, 16 <= n <= 2048
void fft_tables(int n, std::vector<double> &out);            // e^{-i pi k/2n} (n entries) | per-pass twiddle tables
cudaError_t fft_configure();
cudaError_t launch_fft(const FftArgs &a, cudaStream_t stream);

// Seeded uniform[-1,1) white noise, element t a pure function of (seed, offset + t): the input recipe of DESIGN.md §4.
cudaError_t launch_fill_uniform(double *out, size_t count, unsigned long long seed, unsigned long long offset, cudaStream_t stream);

// FP64 pipe microbenchmarks (kind 0: DFMA, 1: DMMA).  Returns TFLOP/s.
cudaError_t run_fp64_peak(int kind, double *tflops);

}  // namespace tpt
