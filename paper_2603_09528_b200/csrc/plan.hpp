// plan.hpp — the plan object behind the opaque tpt_plan handle of include/tpt.h, shared by api.cu and sharded.cu.
#pragma once

#include <cuda_runtime.h>

#include <cstddef>
#include <vector>

#include "../../include/tpt.h"
#include "kernels.cuh"

struct tpt_plan {
    int nx = 0, ny = 0, nz = 0;
    int bc[3] = {0, 0, 0};
    double alpha = 0.0;
    int singular = 0;
    int dirs = TPT_DIRS_XYZ;      // implicitly treated directions: bit 0 = x, 1 = y, 2 = z
    int work_fields = 1;          // fields the workspace holds (tpt_plan_reserve_batch)
    int device = 0;
    double shift0 = 0.0;          // 0 (Poisson) or -1/alpha (Helmholtz, A5)
    int transform[2] = {0, 0};    // per diagonalised direction: TPT_TRANSFORM_GEMM / TPT_TRANSFORM_FFT (uniform directions)
    double fft_s[2][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}};   // [dir]: forward s0, s1, inverse s0, s1 (fft.cu)
    double *d_fft[2] = {nullptr, nullptr};   // twiddle tables
    int gemm_variant = 2;
    int thomas_variant = 1;       // 1 = on-chip partitioned kernel where supported, 0 = streaming kernel
    int slab_groups = -1;         // L2-resident slab pipeline of steps 2.2-2.4: -1 = automatic, 0 = off, G > 0 = slabs of G 16-column groups
    double *d_slab = nullptr;     // its two slab buffers (lazy)
    size_t slab_elems = 0;        // doubles per slab buffer
    cudaStream_t st_slab = nullptr;                    // second stream: odd slabs overlap the even ones
    cudaEvent_t ev_slab_fork = nullptr, ev_slab_join = nullptr;
    // periodic z (A19): Sherman-Morrison around the tridiagonal sweep (kernels.cu launch_cyclic_*)
    int cyclic = 0;
    double cyc_r = 0.0;           // a_0 / g
    double b0_null = 0.0;         // unmodified b_0 (row 0 of the null column)
    double cyc_u[2] = {0.0, 0.0};   // g and c_{n-1}: the right-hand side u of the plan-time sweep
    double *d_cyc_q = nullptr;    // q = A'^-1 u, one field, natural layout (swept at plan time)
    double *d_cyc_rden = nullptr; // 1 / (1 + q_0 + r q_{n-1}) per column
    int fused_small = 1;          // grids that fit on chip: the whole solve in one cluster launch (fused_small.cu)
    int sms = 0;
    int profiling = 0;
    int launches_last = 0;
    std::vector<double> lamx, lamy, qx, qy;   // host copies (inspection)
    // device: pre-scaled transform matrices, all row-major
    double *d_xfwd = nullptr;   // [i][m]  = s * sqrt(wx_i) Q~x[i][m]      B-operand of step 2.1
    double *d_xinv = nullptr;   // [m][i]  = Q~x[i][m] / sqrt(wx_i)         B-operand of step 2.5
    double *d_yfwd = nullptr;   // [m][j]  = sqrt(wy_j) Q~y[j][m]           A-operand of step 2.2
    double *d_yinv = nullptr;   // [j][m]  = Q~y[j][m] / sqrt(wy_j)         A-operand of step 2.4
    double *d_vec = nullptr;    // lamx | lamy | az | bz | cz | wz
    double *d_geo = nullptr;    // rwx | gfx | rwy | gfy | rwz | gfz: 1/width per cell, 1/centre spacing per face (projection.cu)
    tpt::ProjGeom geo{};
    double *d_abc = nullptr;    // coefficient tables of the on-chip Thomas kernel (thomas_onchip_tables)
    double *d_lamx = nullptr, *d_lamy = nullptr, *d_az = nullptr, *d_bz = nullptr, *d_cz = nullptr, *d_wz = nullptr;
    double *d_work = nullptr;   // one field
    double *d_stage = nullptr;  // staging field for tpt_solve_host (lazy)
    // tpt_solve_host pipeline (lazy): copy streams and per-slab events
    cudaStream_t st_h2d = nullptr, st_d2h = nullptr;
    cudaEvent_t ev_start = nullptr, ev_done = nullptr;
    std::vector<cudaEvent_t> ev_slab;   // 2 per z-slab: slab arrived, slab ready to leave
    bool host_ready = false;            // all of the above exist (set last, tpt_solve_host_async)
    // profiling: one set of TPT_K_COUNT+1 events per profiled solve since the last read-out
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;           // events handed out since the last read-out
    long launches_accum = 0;
    size_t points() const { return (size_t)nx * ny * nz; }
};


namespace tpt {
namespace detail {

// Internal pieces of api.cu that the sharded solve (sharded.cu) reuses.
// The transform GEMMs of steps 2.1 / 2.5 (x) and 2.2 / 2.4 (y) on z-planes [k0, k0 + nk) of the fields at in / out.
GemmArgs gemm_x(const tpt_plan *p, const double *in, double *out, const double *mat, int k0, int nk);
GemmArgs gemm_y(const tpt_plan *p, const double *in, double *out, const double *mat, int k0, int nk, bool in_blocked,
                bool out_blocked);
cudaError_t run_gemm(const tpt_plan *p, const GemmArgs &g, cudaStream_t st);
// One transform slot (GEMM or fast transform) on z-planes [k0, k0 + nk); natural layout unless `blocked`.
int run_slot(tpt_plan *p, int slot, const double *in, double *out, cudaStream_t st, int *launches, int k0, int nk,
             bool blocked = false);
bool on_plan_device(const tpt_plan *p);
// tpt_plan_create_ex with a workspace of `work_points` doubles instead of one field (0 = one field)
int plan_create_sized(tpt_plan **plan_out, int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                      const int bc[3], double helmholtz_alpha, int implicit_dirs, const int transform[2], size_t work_points);

}  // namespace detail
}  // namespace tpt
