// api.cu — the C ABI declared in include/tpt.h.  No torch types; plain pointers and sizes.
#include "../../include/tpt.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstring>
#include <deque>
#include <mutex>
#include <new>
#include <vector>

#include "kernels.cuh"
#include "plan.hpp"
#include "plan_host.hpp"

namespace {

int g_eigen_base = 0;   // tpt_debug_set_eigen_base: base eigen-solver of plans created from now on (test only)

// Plan-time eigen-decompositions are O(N^3) host work and depend only on (faces, bc): the last few are kept, so that
// a second plan on the same grid (the two plans of a config-5 step, the e2e double buffer, the P shards of a sharded
// plan in one process) does not repeat them ("reused for every right-hand side").
struct EigenEntry {
    int n, bc, base;
    std::vector<double> faces, lam, q;
};
std::mutex g_eigen_mutex;
std::deque<EigenEntry> g_eigen_cache;

int cached_eigen(const tpt::Operator1D &op, int n, const double *faces, int bc, std::vector<double> &lam, std::vector<double> &q) {
    {
        std::lock_guard<std::mutex> lock(g_eigen_mutex);
        for (const EigenEntry &e : g_eigen_cache)
            if (e.n == n && e.bc == bc && e.base == g_eigen_base && std::memcmp(e.faces.data(), faces, sizeof(double) * (n + 1)) == 0) {
                lam = e.lam;
                q = e.q;
                return 0;
            }
    }
    const int rc = tpt::eigen_decompose(op, lam, q, g_eigen_base);
    if (rc != 0) return rc;
    std::lock_guard<std::mutex> lock(g_eigen_mutex);
    g_eigen_cache.push_front(EigenEntry{n, bc, g_eigen_base, std::vector<double>(faces, faces + n + 1), lam, q});
    if (g_eigen_cache.size() > 4) g_eigen_cache.pop_back();
    return 0;
}

bool bc_valid(int b) { return b == TPT_BC_NEUMANN || b == TPT_BC_DIRICHLET || b == TPT_BC_PERIODIC; }

void free_plan(tpt_plan *p) {
    if (!p) return;
    cudaFree(p->d_xfwd);
    cudaFree(p->d_xinv);
    cudaFree(p->d_yfwd);
    cudaFree(p->d_yinv);
    cudaFree(p->d_vec);
    cudaFree(p->d_abc);
    cudaFree(p->d_geo);
    cudaFree(p->d_fft[0]);
    cudaFree(p->d_fft[1]);
    cudaFree(p->d_work);
    cudaFree(p->d_stage);
    cudaFree(p->d_slab);
    cudaFree(p->d_cyc_q);
    cudaFree(p->d_cyc_rden);
    if (p->ev_slab_fork) cudaEventDestroy(p->ev_slab_fork);
    if (p->ev_slab_join) cudaEventDestroy(p->ev_slab_join);
    if (p->st_slab) cudaStreamDestroy(p->st_slab);
    for (auto &e : p->ev_pool) cudaEventDestroy(e);
    for (auto &e : p->ev_slab) cudaEventDestroy(e);
    if (p->ev_start) cudaEventDestroy(p->ev_start);
    if (p->ev_done) cudaEventDestroy(p->ev_done);
    if (p->st_h2d) cudaStreamDestroy(p->st_h2d);
    if (p->st_d2h) cudaStreamDestroy(p->st_d2h);
    delete p;
}

int upload(double **dst, const std::vector<double> &src) {
    cudaError_t e = cudaMalloc(dst, src.size() * sizeof(double));
    if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorMemoryAllocation ? TPT_ENOMEM : TPT_ECUDA; }
    e = cudaMemcpy(*dst, src.data(), src.size() * sizeof(double), cudaMemcpyHostToDevice);
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

// The transforms act plane by plane in z, so a solve may be issued on z-slabs [k0, k0 + nk) (tpt_solve_host
// overlaps the slabs' copies with their transforms); in / out point at the FIELD, the builders add the slab offset.
tpt::GemmArgs gemm_x(const tpt_plan *p, const double *in, double *out, const double *mat, int k0, int nk) {
    // steps 2.1 / 2.5: all N_y*nk lines at once, out[r][:] = in[r][:] * mat
    const size_t off = (size_t)p->nx * p->ny * k0;
    tpt::GemmArgs g{};
    g.A = in + off; g.B = mat; g.C = out + off;
    g.M = p->ny * nk; g.N = p->nx; g.K = p->nx;
    g.lda = p->nx; g.ldb = p->nx; g.ldc = p->nx;
    g.strideA = g.strideB = g.strideC = 0;
    g.batch = 1;
    return g;
}

// steps 2.2 / 2.4: per z-plane, out_k = mat * in_k  (strided-batched, no transposes).  in_blocked / out_blocked: that
// side is the mode-space field in the tile-blocked layout (kernels.cuh), whose z index has stride 16.
// x0 / ncols: only the columns [x0, x0 + ncols) of every plane (ncols = 0: all); a blocked side is then a slab buffer of
// its own, ncols columns wide (the L2-resident slab pipeline below), a natural side the full field.
tpt::GemmArgs gemm_y(const tpt_plan *p, const double *in, double *out, const double *mat, int k0, int nk,
                     bool in_blocked, bool out_blocked, int x0 = 0, int ncols = 0) {
    const int64_t plane = (int64_t)p->nx * p->ny;
    const int w = ncols ? ncols : p->nx;
    tpt::GemmArgs g{};
    g.A = mat;
    g.M = p->ny; g.N = w; g.K = p->ny;
    g.lda = p->ny; g.strideA = 0;
    g.batch = nk;
    if (in_blocked) { g.B = in + (size_t)16 * k0; g.ldb = (int64_t)w * p->nz; g.strideB = 16; g.ldgB = (int64_t)16 * p->nz; }
    else { g.B = in + (size_t)plane * k0 + x0; g.ldb = p->nx; g.strideB = plane; }
    if (out_blocked) { g.C = out + (size_t)16 * k0; g.ldc = (int64_t)w * p->nz; g.strideC = 16; g.ldgC = (int64_t)16 * p->nz; }
    else { g.C = out + (size_t)plane * k0 + x0; g.ldc = p->nx; g.strideC = plane; }
    return g;
}

// variant 2 = persistent TMA/mbarrier DMMA kernel where the shape allows, else the variant-1 / generic kernels
cudaError_t run_gemm(const tpt_plan *p, const tpt::GemmArgs &g, cudaStream_t st) {
    if (p->gemm_variant == 2 && tpt::gemm_tma_supported(g)) return tpt::launch_gemm_tma(g, p->sms, st);
    if (g.ldgB > 16 || g.ldgC > 16) return cudaErrorInvalidValue;   // only the TMA kernel knows the blocked layout
    return tpt::launch_gemm(g, p->gemm_variant >= 1 ? 1 : 0, st);
}

// The mode-space field (between steps 2.2 and 2.4) is kept tile-blocked when the kernels on both sides of it can:
// the TMA GEMM for the y transforms and the on-chip sweep.  tpt_stage always uses the natural layout.
bool use_blocked(const tpt_plan *p) {
    if (p->thomas_variant != 1 || !(p->dirs & 2) || p->cyclic) return false;   // (the cyclic correction runs in the natural layout)
    if (!tpt::blocked_layout_supported(p->nx, p->ny, p->nz) || !tpt::thomas_onchip_supported(p->nx, p->ny, p->nz)) return false;
    // the fast y transform addresses either layout (its tiles write whole 128-byte lines of the blocked field)
    if (p->transform[1] == TPT_TRANSFORM_FFT) return true;
    return p->gemm_variant == 2 && p->ny % 2 == 0;   // the TMA GEMM (M = K = ny any even size, N = nx a multiple of 16)
}

// Step 2.3 on one field: in -> out (in == out allowed); `scratch` is a free field (used by the streaming kernel only).
int run_sweep(tpt_plan *p, const double *in, double *out, double *scratch, cudaStream_t st, int *launches, bool blocked,
              bool blocked_shape, int singular);

int run_thomas(tpt_plan *p, const double *in, double *out, double *scratch, cudaStream_t st, int *launches, bool blocked = false,
               bool blocked_shape = false) {
    int rc = run_sweep(p, in, out, scratch, st, launches, blocked, blocked_shape, p->singular);
    if (rc != TPT_OK || !p->cyclic) return rc;
    // periodic z: x = y - q (y_0 + r y_{n-1}) rden   (Sherman-Morrison, kernels.cu)
    if (blocked) return TPT_ECUDA;
    ++*launches;
    return tpt::launch_cyclic_correct(out, p->d_cyc_q, p->d_cyc_rden, (size_t)p->nx * p->ny, p->nz, p->cyc_r, st) == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

// the tridiagonal sweep proper (`singular`: treat column (0,0) as the null column)
int run_sweep(tpt_plan *p, const double *in, double *out, double *scratch, cudaStream_t st, int *launches, bool blocked,
              bool blocked_shape, int singular) {
    if (p->thomas_variant == 1 && tpt::thomas_onchip_supported(p->nx, p->ny, p->nz)) {
        // on-chip kernel; the null-mode gauge of a singular plan is fused into it
        cudaError_t e = tpt::launch_thomas_onchip(in, out, p->d_abc, p->d_lamx, p->d_lamy, p->d_wz, p->nx, p->ny, p->nz, p->shift0,
                                                  singular, blocked, blocked_shape, p->sms, st);
        ++*launches;
        return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
    }
    // streaming kernel: in place on `out`, c' spilled to `scratch`; separate gauge kernel
    if (blocked) return TPT_ECUDA;
    if (in != out && cudaMemcpyAsync(out, in, p->points() * sizeof(double), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return TPT_ECUDA;
    cudaError_t e = tpt::launch_thomas(out, scratch, p->d_az, p->d_bz, p->d_cz, p->d_lamx, p->d_lamy, p->nx, p->ny, p->nz,
                                       p->shift0, singular, p->b0_null, st);
    ++*launches;
    if (e == cudaSuccess && singular) {
        e = tpt::launch_gauge(out, p->d_wz, (size_t)p->nx * p->ny, p->nz, st);
        ++*launches;
    }
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

// Runs one transform slot on z-planes [k0, k0 + nk) of the fields at in / out; *launches incremented by the kernels
// enqueued.  `blocked`: the mode-space side of a y transform (output of 2.2, input of 2.4) is tile-blocked.
int run_slot(tpt_plan *p, int slot, const double *in, double *out, cudaStream_t st, int *launches, int k0, int nk,
             bool blocked = false, int x0 = 0, int ncols = 0) {
    cudaError_t e = cudaSuccess;
    const int d = (slot == TPT_K_FWD_X || slot == TPT_K_INV_X) ? 0 : 1;
    if (p->transform[d] == TPT_TRANSFORM_FFT) {   // uniform direction: fast transform, no transposes
        const bool inv = slot == TPT_K_INV_X || slot == TPT_K_INV_Y;
        const size_t off = (size_t)p->nx * p->ny * k0;
        const bool blk = blocked && d == 1;          // mode-space side of a y transform: tile-blocked (offset by k0 inside)
        tpt::FftArgs a{};
        a.in = (blk && inv) ? in : in + off;
        a.out = (blk && !inv) ? out : out + off;
        a.tables = p->d_fft[d];
        a.dir = d; a.inverse = inv ? 1 : 0; a.bc = p->bc[d];
        a.nx = p->nx; a.ny = p->ny; a.planes = nk;
        a.s0 = p->fft_s[d][inv ? 2 : 0]; a.s1 = p->fft_s[d][inv ? 3 : 1];
        a.blocked = blk ? 1 : 0; a.nz = p->nz; a.k0 = k0;
        if (d == 1) { a.x0 = x0; a.ncols = ncols; }
        ++*launches;
        return tpt::launch_fft(a, st) == cudaSuccess ? TPT_OK : TPT_ECUDA;
    }
    switch (slot) {
        case TPT_K_FWD_X: e = run_gemm(p, gemm_x(p, in, out, p->d_xfwd, k0, nk), st); ++*launches; break;
        case TPT_K_INV_X: e = run_gemm(p, gemm_x(p, in, out, p->d_xinv, k0, nk), st); ++*launches; break;
        case TPT_K_FWD_Y: e = run_gemm(p, gemm_y(p, in, out, p->d_yfwd, k0, nk, false, blocked, x0, ncols), st); ++*launches; break;
        case TPT_K_INV_Y: e = run_gemm(p, gemm_y(p, in, out, p->d_yinv, k0, nk, blocked, false, x0, ncols), st); ++*launches; break;
        default: return TPT_EINVAL;
    }
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

bool slot_active(const tpt_plan *p, int slot) {
    if (slot == TPT_K_FWD_X || slot == TPT_K_INV_X) return (p->dirs & 1) != 0;
    if (slot == TPT_K_FWD_Y || slot == TPT_K_INV_Y) return (p->dirs & 2) != 0;
    return slot == TPT_K_THOMAS;
}

// ---- L2-resident slab pipeline of steps 2.2 -> 2.3 -> 2.4 (BASELINE north_star "Fusion") -----------------
// The mode-space field between the forward-y transform, the z sweep and the inverse-y transform is only ever needed one
// x-slab at a time: the y transforms act column by column in x, the sweep column by column in (kx, ky).  So instead of
// writing the whole field to HBM and reading it back twice, the three steps run slab by slab through two small slab
// buffers (G 16-column groups x ny x nz, tile-blocked) that stay resident in the 126 MB L2: 4 of the 10 field-sized HBM
// passes of a solve disappear.  Even and odd slabs alternate between the caller's stream and a second one, so the tail of
// one slab's kernels overlaps the next slab's.  Pays where those steps are HBM-bound (fast y transforms); with GEMM y
// transforms they are FP64-bound and a slab narrow enough for L2 would starve the 128-column GEMM tiles.
size_t slab_bytes(const tpt_plan *p, int groups) { return (size_t)groups * 16 * p->ny * p->nz * sizeof(double); }

int slab_groups_of(const tpt_plan *p) {
    if (!use_blocked(p)) return 0;
    if (p->slab_groups >= 0) return p->slab_groups > p->nx / 16 ? p->nx / 16 : p->slab_groups;
    // automatic: off — measured on the box (profiles/r2_*.md) the slab pipeline does not pay with the present kernels
    return 0;
}

int slab_setup(tpt_plan *p, int groups) {
    const size_t need = slab_bytes(p, groups) / sizeof(double);
    if (p->slab_elems < need) {
        if (cudaDeviceSynchronize() != cudaSuccess) return TPT_ECUDA;
        cudaFree(p->d_slab);
    cudaFree(p->d_cyc_q);
    cudaFree(p->d_cyc_rden);
        p->d_slab = nullptr;
        p->slab_elems = 0;
        cudaError_t e = cudaMalloc(&p->d_slab, 2 * need * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorMemoryAllocation ? TPT_ENOMEM : TPT_ECUDA; }
        p->slab_elems = need;
    }
    if (!p->st_slab) {
        cudaStream_t s2 = nullptr;
        cudaEvent_t ef = nullptr, ej = nullptr;
        if (cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&ef, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ej, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            if (ef) cudaEventDestroy(ef);
            if (ej) cudaEventDestroy(ej);
            if (s2) cudaStreamDestroy(s2);
            return TPT_ECUDA;
        }
        p->st_slab = s2; p->ev_slab_fork = ef; p->ev_slab_join = ej;
    }
    return TPT_OK;
}

// steps 2.2-2.4 of one field, slab by slab: src (natural layout) -> dst (natural layout; src == dst allowed, a slab's
// columns are read completely before they are written)
int run_slabs(tpt_plan *p, const double *src, double *dst, int groups, cudaStream_t st, int *launches) {
    int rc = slab_setup(p, groups);
    if (rc != TPT_OK) return rc;
    const int total = p->nx / 16;
    const int nslabs = (total + groups - 1) / groups;
    const bool two = nslabs > 1;
    if (two && (cudaEventRecord(p->ev_slab_fork, st) != cudaSuccess || cudaStreamWaitEvent(p->st_slab, p->ev_slab_fork, 0) != cudaSuccess))
        return TPT_ECUDA;
    for (int s = 0; s < nslabs; ++s) {
        cudaStream_t q = (s & 1) ? p->st_slab : st;                 // buffer s & 1 belongs to stream s & 1: in-order reuse
        double *buf = p->d_slab + (size_t)(s & 1) * p->slab_elems;
        const int g0 = s * groups, ng = (total - g0 < groups) ? total - g0 : groups;
        const int x0 = g0 * 16, ncols = ng * 16;
        rc = run_slot(p, TPT_K_FWD_Y, src, buf, q, launches, 0, p->nz, true, x0, ncols);
        if (rc != TPT_OK) return rc;
        cudaError_t e = tpt::launch_thomas_onchip(buf, buf, p->d_abc, p->d_lamx + x0, p->d_lamy, p->d_wz, ncols, p->ny, p->nz, p->shift0,
                                                  p->singular && x0 == 0, true, false, p->sms, q);
        ++*launches;
        if (e != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
        rc = run_slot(p, TPT_K_INV_Y, buf, dst, q, launches, 0, p->nz, true, x0, ncols);
        if (rc != TPT_OK) return rc;
    }
    if (two && (cudaEventRecord(p->ev_slab_join, p->st_slab) != cudaSuccess || cudaStreamWaitEvent(st, p->ev_slab_join, 0) != cudaSuccess))
        return TPT_ECUDA;
    return TPT_OK;
}

// Grids that fit on chip run the whole solve as one cluster launch (fused_small.cu) — with the default kernel variants
// only, so that selecting a variant still exercises that kernel.
bool use_fused_small(const tpt_plan *p) {
    if (!p->fused_small || p->gemm_variant != 2 || p->thomas_variant != 1 || p->cyclic) return false;
    if (!(p->dirs & 3)) return false;     // sweep only ("z"): already a single launch
    if (((p->dirs & 1) && p->transform[0] != TPT_TRANSFORM_GEMM) || ((p->dirs & 2) && p->transform[1] != TPT_TRANSFORM_GEMM)) return false;
    return tpt::fused_small_supported(p->nx, p->ny, p->nz);
}

int run_fused_small(tpt_plan *p, const double *rhs, double *out, int nf, cudaStream_t st, int *launches) {
    const size_t pts = p->points();
    for (int f = 0; f < nf; ++f) {
        tpt::FusedSmallArgs a{};
        a.rhs = rhs + f * pts; a.out = out + f * pts; a.work = p->d_work + f * pts;
        a.xfwd = p->d_xfwd; a.xinv = p->d_xinv; a.yfwd = p->d_yfwd; a.yinv = p->d_yinv;
        a.az = p->d_az; a.bz = p->d_bz; a.cz = p->d_cz; a.wz = p->d_wz; a.lamx = p->d_lamx; a.lamy = p->d_lamy;
        a.nx = p->nx; a.ny = p->ny; a.nz = p->nz; a.dirs = p->dirs; a.singular = p->singular; a.shift0 = p->shift0;
        if (tpt::launch_fused_small(a, st) != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
        ++*launches;
    }
    return TPT_OK;
}

// Steps 2.1-2.5 on nf stacked fields (nf <= work_fields).  Buffers: the transforms are out of place and alternate
// between the plan workspace W and `out`, starting with W (rhs may alias out); the sweep works in place on whichever
// holds the data — or straight from rhs to out when no transform is active (the "z" choice of PAPER.md:209) — so the
// result always lands in `out`:  xyz: rhs->W->out->[T]->W->out   yz: rhs->W->[T]->out   z: rhs->[T]->out.
int run_pipeline(tpt_plan *p, const double *rhs, double *out, int nf, cudaStream_t st, cudaEvent_t *ev, int *launches) {
    const double *cur = rhs;
    double *W = p->d_work;
    const size_t pts = p->points();
    const int nk = p->nz * nf;
    const bool blk = use_blocked(p);
    if (ev && cudaEventRecord(ev[0], st) != cudaSuccess) return TPT_ECUDA;
    if (use_fused_small(p)) {      // one launch: its time is reported in the first slot
        int rc = run_fused_small(p, rhs, out, nf, st, launches);
        if (rc != TPT_OK) return rc;
        for (int s = 0; ev && s < TPT_K_COUNT; ++s)
            if (cudaEventRecord(ev[s + 1], st) != cudaSuccess) return TPT_ECUDA;
        return TPT_OK;
    }
    const int slabs = slab_groups_of(p);
    if (slabs > 0) {
        // xyz: rhs -> W (2.1) -> slabs: W -> W (2.2-2.4) -> out (2.5);   yz: slabs: rhs -> out
        const bool use_x = (p->dirs & 1) != 0;
        int rc = TPT_OK;
        if (use_x) rc = run_slot(p, TPT_K_FWD_X, rhs, W, st, launches, 0, nk);
        if (rc != TPT_OK) return rc;
        if (ev && cudaEventRecord(ev[TPT_K_FWD_X + 1], st) != cudaSuccess) return TPT_ECUDA;
        for (int f = 0; f < nf && rc == TPT_OK; ++f)
            rc = run_slabs(p, (use_x ? W : rhs) + f * pts, (use_x ? W : out) + f * pts, slabs, st, launches);
        if (rc != TPT_OK) return rc;
        // the three steps interleave slab by slab: their time is reported in the forward-y slot
        for (int s = TPT_K_FWD_Y; ev && s <= TPT_K_INV_Y; ++s)
            if (cudaEventRecord(ev[s + 1], st) != cudaSuccess) return TPT_ECUDA;
        if (use_x) rc = run_slot(p, TPT_K_INV_X, W, out, st, launches, 0, nk);
        if (rc != TPT_OK) return rc;
        if (ev && cudaEventRecord(ev[TPT_K_INV_X + 1], st) != cudaSuccess) return TPT_ECUDA;
        return TPT_OK;
    }
    for (int s = 0; s < TPT_K_COUNT; ++s) {
        int rc = TPT_OK;
        if (s == TPT_K_THOMAS) {
            double *dst = (cur == rhs) ? out : const_cast<double *>(cur);
            double *scratch = (dst == W) ? out : W;
            for (int f = 0; f < nf && rc == TPT_OK; ++f)
                rc = run_thomas(p, cur + f * pts, dst + f * pts, scratch + f * pts, st, launches, blk);
            cur = dst;
        } else if (slot_active(p, s)) {
            double *dst = (cur == W) ? out : W;
            if (blk && (s == TPT_K_FWD_Y || s == TPT_K_INV_Y)) {   // the blocked layout is per field: one launch each
                for (int f = 0; f < nf && rc == TPT_OK; ++f)
                    rc = run_slot(p, s, cur + f * pts, dst + f * pts, st, launches, 0, p->nz, true);
            } else {
                rc = run_slot(p, s, cur, dst, st, launches, 0, nk);   // the stack is just a longer z axis
            }
            cur = dst;
        }
        if (rc != TPT_OK) return rc;
        if (ev && cudaEventRecord(ev[s + 1], st) != cudaSuccess) return TPT_ECUDA;
    }
    return cur == out ? TPT_OK : TPT_ECUDA;
}

bool aligned16(const void *q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; }
bool aligned8(const void *q) { return (reinterpret_cast<uintptr_t>(q) & 7) == 0; }

// tpt.h: "the same device must be current in later calls on that plan" — a launch on another device would read the
// plan's matrices through an invalid context; refuse instead.
bool on_plan_device(const tpt_plan *p) {
    int d = -1;
    if (cudaGetDevice(&d) != cudaSuccess) { cudaGetLastError(); return false; }
    return d == p->device;
}

}  // namespace

namespace tpt {
namespace detail {
GemmArgs gemm_x(const tpt_plan *p, const double *in, double *out, const double *mat, int k0, int nk) {
    return ::gemm_x(p, in, out, mat, k0, nk);
}
GemmArgs gemm_y(const tpt_plan *p, const double *in, double *out, const double *mat, int k0, int nk, bool in_blocked,
                bool out_blocked) {
    return ::gemm_y(p, in, out, mat, k0, nk, in_blocked, out_blocked, 0, 0);
}
cudaError_t run_gemm(const tpt_plan *p, const GemmArgs &g, cudaStream_t st) { return ::run_gemm(p, g, st); }
int run_slot(tpt_plan *p, int slot, const double *in, double *out, cudaStream_t st, int *launches, int k0, int nk, bool blocked) {
    return ::run_slot(p, slot, in, out, st, launches, k0, nk, blocked, 0, 0);
}
bool on_plan_device(const tpt_plan *p) { return ::on_plan_device(p); }
}  // namespace detail
}  // namespace tpt

extern "C" {

int tpt_plan_create(tpt_plan **plan_out, int nx, int ny, int nz, const double *xf, const double *yf,
                    const double *zf, const int bc[3], double helmholtz_alpha) {
    return tpt_plan_create_dirs(plan_out, nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha, TPT_DIRS_XYZ);
}

int tpt_plan_create_dirs(tpt_plan **plan_out, int nx, int ny, int nz, const double *xf, const double *yf,
                         const double *zf, const int bc[3], double helmholtz_alpha, int implicit_dirs) {
    const int gemm[2] = {TPT_TRANSFORM_GEMM, TPT_TRANSFORM_GEMM};
    return tpt_plan_create_ex(plan_out, nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha, implicit_dirs, gemm);
}

// uniform to rounding: every width within a few ulps of the coordinate scale of (x_n - x_0) / n
static bool direction_uniform(int n, const double *f) {
    const double d = (f[n] - f[0]) / n;
    const double tol = 16.0 * 2.220446049250313e-16 * std::fmax(std::fabs(f[0]), std::fabs(f[n]));
    for (int i = 0; i < n; ++i)
        if (std::fabs((f[i + 1] - f[i]) - d) > tol) return false;
    return true;
}

int tpt_plan_create_ex(tpt_plan **plan_out, int nx, int ny, int nz, const double *xf, const double *yf,
                       const double *zf, const int bc[3], double helmholtz_alpha, int implicit_dirs, const int transform[2]) {
    return tpt::detail::plan_create_sized(plan_out, nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha, implicit_dirs, transform, 0);
}

}  // extern "C"

int tpt::detail::plan_create_sized(tpt_plan **plan_out, int nx, int ny, int nz, const double *xf, const double *yf,
                                   const double *zf, const int bc[3], double helmholtz_alpha, int implicit_dirs,
                                   const int transform[2], size_t work_points) {
    if (!plan_out || !bc || !transform) return TPT_EINVAL;
    for (int d = 0; d < 2; ++d)
        if (transform[d] != TPT_TRANSFORM_GEMM && transform[d] != TPT_TRANSFORM_FFT) return TPT_EINVAL;
    if (implicit_dirs != TPT_DIRS_XYZ && implicit_dirs != TPT_DIRS_YZ && implicit_dirs != TPT_DIRS_Z) return TPT_EINVAL;
    if (implicit_dirs != TPT_DIRS_XYZ && !(helmholtz_alpha > 0.0)) return TPT_EINVAL;   // Eq. 2c carries the full L
    if (!tpt::faces_valid(nx, xf) || !tpt::faces_valid(ny, yf) || !tpt::faces_valid(nz, zf)) return TPT_EINVAL;
    if (!bc_valid(bc[0]) || !bc_valid(bc[1]) || !bc_valid(bc[2])) return TPT_EINVAL;
    // periodic x, y are diagonalised; a periodic z makes the sweep cyclic (A19)
    if ((bc[2] == TPT_BC_PERIODIC && nz < 3) || (bc[0] == TPT_BC_PERIODIC && nx < 3) || (bc[1] == TPT_BC_PERIODIC && ny < 3)) return TPT_EINVAL;
    if (!(helmholtz_alpha >= 0.0) || !std::isfinite(helmholtz_alpha)) return TPT_EINVAL;
    if ((double)nx * ny * nz > 4.0e9) return TPT_EINVAL;
    // fast transforms: diagonalised, uniform, power-of-two directions only; y tiles need nx % 16 == 0
    if (transform[0] == TPT_TRANSFORM_FFT &&
        (!(implicit_dirs & 1) || !tpt::fft_supported(nx) || !direction_uniform(nx, xf))) return TPT_EINVAL;
    if (transform[1] == TPT_TRANSFORM_FFT &&
        (!(implicit_dirs & 2) || !tpt::fft_supported(ny) || !direction_uniform(ny, yf) || nx % 16)) return TPT_EINVAL;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
    int cc_major = 0;
    if (cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        return TPT_ECUDA;
    }
    if (cc_major != 10) return TPT_ECUDA;   // sm_100a binary only; no fallback
    int sm_count = 0;
    if (cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sm_count < 1) {
        cudaGetLastError();
        return TPT_ECUDA;
    }

    tpt_plan *p = new (std::nothrow) tpt_plan();
    if (!p) return TPT_ENOMEM;
    p->nx = nx; p->ny = ny; p->nz = nz;
    p->bc[0] = bc[0]; p->bc[1] = bc[1]; p->bc[2] = bc[2];
    p->alpha = helmholtz_alpha;
    p->dirs = implicit_dirs;
    p->transform[0] = transform[0]; p->transform[1] = transform[1];
    p->device = dev;
    p->sms = sm_count;
    p->singular = (helmholtz_alpha == 0.0 && bc[0] != TPT_BC_DIRICHLET && bc[1] != TPT_BC_DIRICHLET &&
                   bc[2] != TPT_BC_DIRICHLET) ? 1 : 0;
    p->cyclic = bc[2] == TPT_BC_PERIODIC ? 1 : 0;
    // Helmholtz (I - alpha T) u = f  <=>  (T - I/alpha) u = -f/alpha: same z kernel with a constant
    // extra shift, the -1/alpha scale folded into the first forward matrix ("constant shift").
    // With no transform at all (the "z" choice) the sweep solves (I - alpha T_z) u = f on scaled coefficients.
    const bool use_x = (implicit_dirs & 1) != 0, use_y = (implicit_dirs & 2) != 0;
    const bool z_only = !use_x && !use_y;
    const double rhs_scale = helmholtz_alpha > 0.0 ? -1.0 / helmholtz_alpha : 1.0;
    const double x_scale = use_x ? rhs_scale : 1.0, y_scale = use_x ? 1.0 : rhs_scale;
    p->shift0 = (helmholtz_alpha > 0.0 && !z_only) ? -1.0 / helmholtz_alpha : 0.0;

    int rc = TPT_OK;
    try {
        tpt::Operator1D ox, oy, oz;
        tpt::build_operator(nx, xf, bc[0], ox);
        tpt::build_operator(ny, yf, bc[1], oy);
        tpt::build_operator(nz, zf, bc[2], oz);
        if (z_only) {   // (I - alpha T_z): sub/diag/super = -alpha a, 1 - alpha b, -alpha c
            for (int k = 0; k < nz; ++k) {
                oz.a[k] *= -helmholtz_alpha;
                oz.b[k] = 1.0 - helmholtz_alpha * oz.b[k];
                oz.c[k] *= -helmholtz_alpha;
            }
        }
        // Periodic z: the sweep kernels solve the tridiagonal A' = A - u v^T (corners b_0 - g and b_{n-1} - c_{n-1} a_0 / g with
        // g = -b_0, which only strengthens the diagonal); the rank-one term is put back after the sweep (run_thomas).  The
        // null column of a singular plan keeps the unmodified diagonal: with x_{n-1} = 0 both corner
        // couplings vanish.
        std::vector<double> bz_null;
        double cyc_g = 0.0, cyc_cn = 0.0;
        p->b0_null = oz.b[0];
        if (p->cyclic) {
            bz_null = oz.b;
            cyc_g = -oz.b[0];
            cyc_cn = oz.c[nz - 1];
            p->cyc_r = oz.a[0] / cyc_g;
            oz.b[0] -= cyc_g;
            oz.b[nz - 1] -= cyc_cn * oz.a[0] / cyc_g;
            oz.a[0] = 0.0;
            oz.c[nz - 1] = 0.0;
        }
        // a direction that is not diagonalised contributes no modal shift (Eq. 9 restricted)
        p->lamx.assign(nx, 0.0);
        p->lamy.assign(ny, 0.0);
        const bool fx = use_x && transform[0] == TPT_TRANSFORM_FFT, fy = use_y && transform[1] == TPT_TRANSFORM_FFT;
        // uniform direction with a fast transform: analytical eigenvalues, closed-form basis of fft.cu;
        // the operator is the exactly uniform one with spacing (x_n - x_0) / n
        auto setup_fft = [&](int d, int n, const double *f, int b, double scale, std::vector<double> &lam) {
            const long double pi = 3.14159265358979323846264338327950288L;
            const double dl = (f[n] - f[0]) / n;
            for (int slot = 0; slot < n; ++slot) {
                const long double arg = b == TPT_BC_NEUMANN ? pi * slot / (2.0L * n)
                                      : b == TPT_BC_DIRICHLET ? pi * (slot + 1) / (2.0L * n) : pi * ((slot + 1) / 2) / (long double)n;
                const long double sn = sinl(arg);
                lam[slot] = (double)(-4.0L * sn * sn / ((long double)dl * dl));
            }
            p->fft_s[d][0] = scale * std::sqrt(dl) * std::sqrt(1.0 / n);
            p->fft_s[d][1] = scale * std::sqrt(dl) * std::sqrt(2.0 / n);
            p->fft_s[d][2] = std::sqrt(1.0 / n) / std::sqrt(dl);
            p->fft_s[d][3] = std::sqrt(2.0 / n) / std::sqrt(dl);
            std::vector<double> t;
            tpt::fft_tables(n, t);
            return upload(&p->d_fft[d], t);
        };
        if (fx) rc = setup_fft(0, nx, xf, bc[0], x_scale, p->lamx);
        if (rc == TPT_OK && fy) rc = setup_fft(1, ny, yf, bc[1], y_scale, p->lamy);
        if (rc == TPT_OK && use_x && !fx && cached_eigen(ox, nx, xf, bc[0], p->lamx, p->qx) != 0) rc = TPT_ENUMERIC;
        if (rc == TPT_OK && use_y && !fy) {
            bool same = (use_x && !fx && nx == ny && bc[0] == bc[1] && std::memcmp(xf, yf, sizeof(double) * (nx + 1)) == 0);
            if (same) { p->lamy = p->lamx; p->qy = p->qx; }
            else if (cached_eigen(oy, ny, yf, bc[1], p->lamy, p->qy) != 0) rc = TPT_ENUMERIC;
        }
        if (rc == TPT_OK && use_x && !fx) {
            std::vector<double> m((size_t)nx * nx);
            for (int i = 0; i < nx; ++i) {
                const double s = x_scale * std::sqrt(ox.w[i]);
                for (int k = 0; k < nx; ++k) m[(size_t)i * nx + k] = s * p->qx[(size_t)i * nx + k];
            }
            rc = upload(&p->d_xfwd, m);
            if (rc == TPT_OK) {
                for (int i = 0; i < nx; ++i) {
                    const double s = 1.0 / std::sqrt(ox.w[i]);
                    for (int k = 0; k < nx; ++k) m[(size_t)k * nx + i] = s * p->qx[(size_t)i * nx + k];
                }
                rc = upload(&p->d_xinv, m);
            }
        }
        if (rc == TPT_OK && use_y && !fy) {
            std::vector<double> m((size_t)ny * ny, 0.0);
            if (rc == TPT_OK) {
                for (int j = 0; j < ny; ++j) {
                    const double s = y_scale * std::sqrt(oy.w[j]);
                    for (int k = 0; k < ny; ++k) m[(size_t)k * ny + j] = s * p->qy[(size_t)j * ny + k];
                }
                rc = upload(&p->d_yfwd, m);
            }
            if (rc == TPT_OK) {
                for (int j = 0; j < ny; ++j) {
                    const double s = 1.0 / std::sqrt(oy.w[j]);
                    for (int k = 0; k < ny; ++k) m[(size_t)j * ny + k] = s * p->qy[(size_t)j * ny + k];
                }
                rc = upload(&p->d_yinv, m);
            }
        }
        if (rc == TPT_OK) {
            std::vector<double> v;
            v.reserve((size_t)nx + ny + 4 * (size_t)nz + 8);
            auto pad2 = [&]() { if (v.size() & 1) v.push_back(0.0); };
            size_t o_lamx = v.size(); v.insert(v.end(), p->lamx.begin(), p->lamx.end()); pad2();
            size_t o_lamy = v.size(); v.insert(v.end(), p->lamy.begin(), p->lamy.end()); pad2();
            size_t o_az = v.size(); v.insert(v.end(), oz.a.begin(), oz.a.end()); pad2();
            size_t o_bz = v.size(); v.insert(v.end(), oz.b.begin(), oz.b.end()); pad2();
            size_t o_cz = v.size(); v.insert(v.end(), oz.c.begin(), oz.c.end()); pad2();
            size_t o_wz = v.size(); v.insert(v.end(), oz.w.begin(), oz.w.end()); pad2();
            rc = upload(&p->d_vec, v);
            p->d_lamx = p->d_vec + o_lamx; p->d_lamy = p->d_vec + o_lamy;
            p->d_az = p->d_vec + o_az; p->d_bz = p->d_vec + o_bz; p->d_cz = p->d_vec + o_cz; p->d_wz = p->d_vec + o_wz;
        }
        if (rc == TPT_OK) {   // geometry of the staggered divergence / gradient (Eq. 2c-2e)
            std::vector<double> v;
            size_t off[6];
            const tpt::Operator1D *ops[3] = {&ox, &oy, &oz};
            for (int d = 0; d < 3; ++d) {
                off[2 * d] = v.size();
                for (double wd : ops[d]->w) v.push_back(1.0 / wd);
                if (v.size() & 1) v.push_back(0.0);
                off[2 * d + 1] = v.size();
                for (double dl : ops[d]->delta) v.push_back(1.0 / dl);
                if (v.size() & 1) v.push_back(0.0);
            }
            rc = upload(&p->d_geo, v);
            p->geo.nx = nx; p->geo.ny = ny; p->geo.nz = nz;
            for (int d = 0; d < 3; ++d) p->geo.bc[d] = bc[d];
            p->geo.rwx = p->d_geo + off[0]; p->geo.gfx = p->d_geo + off[1];
            p->geo.rwy = p->d_geo + off[2]; p->geo.gfy = p->d_geo + off[3];
            p->geo.rwz = p->d_geo + off[4]; p->geo.gfz = p->d_geo + off[5];
        }
        if (rc == TPT_OK) {
            std::vector<double> t;
            tpt::thomas_onchip_tables(nz, oz.a.data(), oz.b.data(), oz.c.data(), t, p->cyclic ? bz_null.data() : nullptr);
            rc = upload(&p->d_abc, t);
        }
        if (rc == TPT_OK && p->cyclic) {
            cudaError_t e = cudaMalloc(&p->d_cyc_q, p->points() * sizeof(double));
            if (e == cudaSuccess) e = cudaMalloc(&p->d_cyc_rden, (size_t)nx * ny * sizeof(double));
            if (e != cudaSuccess) { cudaGetLastError(); rc = e == cudaErrorMemoryAllocation ? TPT_ENOMEM : TPT_ECUDA; }
            p->cyc_u[0] = cyc_g; p->cyc_u[1] = cyc_cn;
        }
    } catch (const std::bad_alloc &) {
        rc = TPT_ENOMEM;
    } catch (...) {
        rc = TPT_ECUDA;
    }
    if (rc == TPT_OK) {
        cudaError_t e = cudaMalloc(&p->d_work, (work_points ? work_points : p->points()) * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); rc = (e == cudaErrorMemoryAllocation) ? TPT_ENOMEM : TPT_ECUDA; }
    }
    if (rc == TPT_OK && (tpt::gemm_configure() != cudaSuccess || tpt::gemm_tma_configure() != cudaSuccess ||
                         tpt::fft_configure() != cudaSuccess)) {
        cudaGetLastError();
        rc = TPT_ECUDA;
    }
    if (rc == TPT_OK && p->cyclic) {
        // q = A'^-1 u for every column (its spectral shift is all that distinguishes the columns): one sweep at plan time
        int launches = 0;
        const size_t cols = (size_t)nx * ny;
        cudaError_t e = tpt::launch_cyclic_rhs(p->d_cyc_q, cols, nz, p->cyc_u[0], p->cyc_u[1], nullptr);
        if (e == cudaSuccess) rc = run_sweep(p, p->d_cyc_q, p->d_cyc_q, p->d_work, nullptr, &launches, false, false, 0);
        if (e == cudaSuccess && rc == TPT_OK) e = tpt::launch_cyclic_rden(p->d_cyc_q, p->d_cyc_rden, cols, nz, p->cyc_r, p->singular, nullptr);
        if (e == cudaSuccess && rc == TPT_OK) e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { cudaGetLastError(); rc = TPT_ECUDA; }
    }
    if (rc != TPT_OK) { free_plan(p); return rc; }
    *plan_out = p;
    return TPT_OK;
}

extern "C" {

int tpt_solve(tpt_plan *p, const double *rhs_dev, double *out_dev, void *cuda_stream) {
    if (!p || !rhs_dev || !out_dev || !aligned16(rhs_dev) || !aligned16(out_dev) || !on_plan_device(p)) return TPT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0;
    const bool prof = p->profiling != 0;
    cudaEvent_t *ev = nullptr;
    if (prof) {
        const size_t need = p->ev_used + TPT_K_COUNT + 1;
        if (need > 4096 * (TPT_K_COUNT + 1)) return TPT_EINVAL;   // read the times out first
        try {
            while (p->ev_pool.size() < need) {
                cudaEvent_t e;
                if (cudaEventCreate(&e) != cudaSuccess) return TPT_ECUDA;
                p->ev_pool.push_back(e);
            }
        } catch (const std::bad_alloc &) { return TPT_ENOMEM; }
        ev = p->ev_pool.data() + p->ev_used;
        p->ev_used = need;
    }
    int rc = run_pipeline(p, rhs_dev, out_dev, 1, st, ev, &launches);
    if (rc != TPT_OK) return rc;
    p->launches_last = launches;
    if (prof) p->launches_accum += launches;
    return TPT_OK;
}

// The one-launch solve of fused_small.cu with its scratch in a static device array: no allocation on this call path
// (no cudaMalloc / cudaFree / event or stream creation; the plan's workspace and profiling events are not touched).
int tpt_solve_static_scratch(tpt_plan *p, const double *rhs_dev, double *out_dev, void *cuda_stream) {
    if (!p || !rhs_dev || !out_dev || !aligned16(rhs_dev) || !aligned16(out_dev) || !on_plan_device(p)) return TPT_EINVAL;
    if (p->points() > (size_t)TPT_STATIC_SCRATCH_POINTS) return TPT_ELIMIT;
    // what the fused kernel computes: GEMM transforms in at least one direction, tridiagonal (non-periodic) z
    if (p->cyclic || !(p->dirs & 3)) return TPT_EINVAL;
    if (((p->dirs & 1) && p->transform[0] != TPT_TRANSFORM_GEMM) || ((p->dirs & 2) && p->transform[1] != TPT_TRANSFORM_GEMM)) return TPT_EINVAL;
    if (!tpt::fused_small_supported(p->nx, p->ny, p->nz)) return TPT_ELIMIT;
    tpt::FusedSmallArgs a{};
    a.rhs = rhs_dev; a.out = out_dev; a.work = nullptr;
    a.xfwd = p->d_xfwd; a.xinv = p->d_xinv; a.yfwd = p->d_yfwd; a.yinv = p->d_yinv;
    a.az = p->d_az; a.bz = p->d_bz; a.cz = p->d_cz; a.wz = p->d_wz; a.lamx = p->d_lamx; a.lamy = p->d_lamy;
    a.nx = p->nx; a.ny = p->ny; a.nz = p->nz; a.dirs = p->dirs; a.singular = p->singular; a.shift0 = p->shift0;
    if (tpt::launch_fused_small_static(a, static_cast<cudaStream_t>(cuda_stream)) != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
    p->launches_last = 1;
    return TPT_OK;
}

int tpt_plan_reserve_batch(tpt_plan *p, int nrhs) {
    if (!p || nrhs < 1 || (double)nrhs * (double)p->points() > 8.0e9 || !on_plan_device(p)) return TPT_EINVAL;
    if (nrhs <= p->work_fields) return TPT_OK;
    if (cudaDeviceSynchronize() != cudaSuccess) return TPT_ECUDA;
    double *w = nullptr;
    cudaError_t e = cudaMalloc(&w, (size_t)nrhs * p->points() * sizeof(double));
    if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorMemoryAllocation ? TPT_ENOMEM : TPT_ECUDA; }
    cudaFree(p->d_work);
    p->d_work = w;
    p->work_fields = nrhs;
    return TPT_OK;
}

int tpt_solve_batch(tpt_plan *p, const double *rhs_dev, double *out_dev, int nrhs, void *cuda_stream) {
    if (!p || !rhs_dev || !out_dev || nrhs < 1 || !aligned16(rhs_dev) || !aligned16(out_dev) || !on_plan_device(p)) return TPT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0;
    const size_t pts = p->points();
    for (int f0 = 0; f0 < nrhs; f0 += p->work_fields) {
        const int nf = nrhs - f0 < p->work_fields ? nrhs - f0 : p->work_fields;
        int rc = run_pipeline(p, rhs_dev + (size_t)f0 * pts, out_dev + (size_t)f0 * pts, nf, st, nullptr, &launches);
        if (rc != TPT_OK) return rc;
    }
    p->launches_last = launches;
    return TPT_OK;
}

// z-slabs of a host solve: about 32 MiB each, at most 16 (the transforms of a slab hide under the next slab's copy)
static int host_slabs(const tpt_plan *p) {
    const size_t bytes = p->points() * sizeof(double);
    size_t n = bytes / ((size_t)32 << 20);
    if (n < 1) n = 1;
    if (n > 16) n = 16;
    if (n > (size_t)p->nz) n = (size_t)p->nz;
    return (int)n;
}

int tpt_solve_host(tpt_plan *p, const double *rhs_host, double *out_host, void *cuda_stream) {
    int rc = tpt_solve_host_async(p, rhs_host, out_host, cuda_stream);
    return rc == TPT_OK ? tpt_plan_wait(p) : rc;
}

int tpt_plan_wait(tpt_plan *p) {
    if (!p) return TPT_EINVAL;
    if (!p->host_ready) return TPT_OK;   // no host solve was ever enqueued
    return cudaEventSynchronize(p->ev_done) == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

int tpt_solve_host_async(tpt_plan *p, const double *rhs_host, double *out_host, void *cuda_stream) {
    if (!p || !rhs_host || !out_host || !on_plan_device(p)) return TPT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t bytes = p->points() * sizeof(double);
    if (!p->d_stage) {
        cudaError_t e = cudaMalloc(&p->d_stage, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); p->d_stage = nullptr; return e == cudaErrorMemoryAllocation ? TPT_ENOMEM : TPT_ECUDA; }
    }
    const int ns = host_slabs(p);
    if (!p->host_ready) {
        // every stream and event is created into locals and committed to the plan only when all of them exist: a
        // partial failure leaves the plan as it was (no null stream silently becoming the legacy default stream)
        cudaStream_t s_in = nullptr, s_out = nullptr;
        cudaEvent_t e_start = nullptr, e_done = nullptr;
        std::vector<cudaEvent_t> slab;
        bool ok = true;
        try { slab.assign(2 * 16, nullptr); } catch (const std::bad_alloc &) { return TPT_ENOMEM; }
        ok = cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking) == cudaSuccess &&
             cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking) == cudaSuccess &&
             cudaEventCreateWithFlags(&e_start, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&e_done, cudaEventDisableTiming) == cudaSuccess;
        for (size_t q = 0; ok && q < slab.size(); ++q) ok = cudaEventCreateWithFlags(&slab[q], cudaEventDisableTiming) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();
            for (auto &e : slab) if (e) cudaEventDestroy(e);
            if (e_start) cudaEventDestroy(e_start);
            if (e_done) cudaEventDestroy(e_done);
            if (s_in) cudaStreamDestroy(s_in);
            if (s_out) cudaStreamDestroy(s_out);
            return TPT_ECUDA;
        }
        p->st_h2d = s_in; p->st_d2h = s_out; p->ev_start = e_start; p->ev_done = e_done;
        p->ev_slab.swap(slab);
        p->host_ready = true;
    }
    // Slab pipeline: the transforms act plane by plane, so slab s is transformed (2.1, 2.2) while slab s+1 is still
    // on the bus; after the sweep (which needs every plane) slab s leaves while slab s+1 is transformed back.
    const size_t plane = (size_t)p->nx * p->ny;
    auto k_lo = [&](int s) { return (int)((long long)p->nz * s / ns); };
    int launches = 0;
    if (cudaEventRecord(p->ev_start, st) != cudaSuccess) return TPT_ECUDA;          // order after earlier work on st
    if (cudaStreamWaitEvent(p->st_h2d, p->ev_start, 0) != cudaSuccess) return TPT_ECUDA;
    // buffers alternate between the staging field and the workspace, as in run_pipeline
    double *const S = p->d_stage, *const W = p->d_work;
    const int fwd[2] = {TPT_K_FWD_X, TPT_K_FWD_Y}, inv[2] = {TPT_K_INV_Y, TPT_K_INV_X};
    double *cur = S;
    // natural layout throughout: the tile-blocked mode-space layout scatters a slab's output over the whole field,
    // which here would overwrite later slabs still waiting in the same buffers (and the path is PCIe-bound anyway)
    const bool blk = false;
    for (int s = 0; s < ns; ++s) {
        const int k0 = k_lo(s), nk = k_lo(s + 1) - k0;
        const size_t off = plane * k0, cnt = plane * nk;
        if (cudaMemcpyAsync(S + off, rhs_host + off, cnt * sizeof(double), cudaMemcpyHostToDevice, p->st_h2d) != cudaSuccess ||
            cudaEventRecord(p->ev_slab[2 * s], p->st_h2d) != cudaSuccess ||
            cudaStreamWaitEvent(st, p->ev_slab[2 * s], 0) != cudaSuccess)
            return TPT_ECUDA;
        cur = S;
        for (int q = 0; q < 2; ++q) {
            if (!slot_active(p, fwd[q])) continue;
            double *dst = cur == S ? W : S;
            int rc = run_slot(p, fwd[q], cur, dst, st, &launches, k0, nk, blk);
            if (rc != TPT_OK) return rc;
            cur = dst;
        }
    }
    int rc = run_thomas(p, cur, cur, cur == S ? W : S, st, &launches, blk, use_blocked(p));   // same partition as tpt_solve
    if (rc != TPT_OK) return rc;
    double *const mid = cur;
    for (int s = 0; s < ns; ++s) {
        const int k0 = k_lo(s), nk = k_lo(s + 1) - k0;
        const size_t off = plane * k0, cnt = plane * nk;
        cur = mid;
        for (int q = 0; q < 2; ++q) {
            if (!slot_active(p, inv[q])) continue;
            double *dst = cur == S ? W : S;
            rc = run_slot(p, inv[q], cur, dst, st, &launches, k0, nk, blk);
            if (rc != TPT_OK) return rc;
            cur = dst;
        }
        if (cudaEventRecord(p->ev_slab[2 * s + 1], st) != cudaSuccess ||
            cudaStreamWaitEvent(p->st_d2h, p->ev_slab[2 * s + 1], 0) != cudaSuccess ||
            cudaMemcpyAsync(out_host + off, cur + off, cnt * sizeof(double), cudaMemcpyDeviceToHost, p->st_d2h) != cudaSuccess)
            return TPT_ECUDA;
    }
    if (cudaEventRecord(p->ev_done, p->st_d2h) != cudaSuccess || cudaStreamWaitEvent(st, p->ev_done, 0) != cudaSuccess)
        return TPT_ECUDA;
    p->launches_last = launches;
    return TPT_OK;
}

int tpt_divergence(tpt_plan *p, const double *u_dev, const double *v_dev, const double *w_dev, double scale, double *out_dev,
                   void *cuda_stream) {
    if (!p || !u_dev || !v_dev || !w_dev || !out_dev || !std::isfinite(scale) || !on_plan_device(p)) return TPT_EINVAL;
    if (!aligned8(u_dev) || !aligned8(v_dev) || !aligned8(w_dev) || !aligned8(out_dev)) return TPT_EINVAL;
    cudaError_t e = tpt::launch_divergence(u_dev, v_dev, w_dev, p->geo, scale, out_dev, static_cast<cudaStream_t>(cuda_stream));
    p->launches_last = 1;
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

static bool dirs_valid(int d) { return d == TPT_DIRS_XYZ || d == TPT_DIRS_YZ || d == TPT_DIRS_Z; }

int tpt_gradient_correct(tpt_plan *p, const double *phi_dev, double c, double *u_dev, double *v_dev, double *w_dev, double *p_dev,
                         double alpha_p, int implicit_dirs, void *cuda_stream) {
    if (!p || !phi_dev || !u_dev || !v_dev || !w_dev || !std::isfinite(c) || !on_plan_device(p)) return TPT_EINVAL;
    if (!aligned8(phi_dev) || !aligned8(u_dev) || !aligned8(v_dev) || !aligned8(w_dev) || !aligned8(p_dev)) return TPT_EINVAL;
    if (p_dev && (!(alpha_p >= 0.0) || !std::isfinite(alpha_p) || !dirs_valid(implicit_dirs))) return TPT_EINVAL;
    cudaError_t e = tpt::launch_correct(phi_dev, u_dev, v_dev, w_dev, p_dev, p->geo, c, alpha_p, implicit_dirs,
                                        static_cast<cudaStream_t>(cuda_stream));
    p->launches_last = 1;
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

int tpt_project(tpt_plan *p, double *u_dev, double *v_dev, double *w_dev, double gamma_dt, double *phi_dev, double *p_dev,
                double alpha_p, int implicit_dirs, void *cuda_stream) {
    if (!p || !u_dev || !v_dev || !w_dev || !phi_dev || !aligned16(phi_dev) || !on_plan_device(p)) return TPT_EINVAL;
    if (!aligned8(u_dev) || !aligned8(v_dev) || !aligned8(w_dev) || !aligned8(p_dev)) return TPT_EINVAL;
    if (p->alpha != 0.0 || p->dirs != TPT_DIRS_XYZ) return TPT_EINVAL;       // Eq. 2c carries the full Laplacian
    if (!(gamma_dt > 0.0) || !std::isfinite(gamma_dt)) return TPT_EINVAL;
    if (p_dev && (!(alpha_p >= 0.0) || !std::isfinite(alpha_p) || !dirs_valid(implicit_dirs))) return TPT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (tpt::launch_divergence(u_dev, v_dev, w_dev, p->geo, 1.0 / gamma_dt, phi_dev, st) != cudaSuccess) return TPT_ECUDA;
    int rc = tpt_solve(p, phi_dev, phi_dev, cuda_stream);                      // in place: rhs -> Phi
    if (rc != TPT_OK) return rc;
    const int solve_launches = p->launches_last;
    if (tpt::launch_correct(phi_dev, u_dev, v_dev, w_dev, p_dev, p->geo, gamma_dt, alpha_p, implicit_dirs, st) != cudaSuccess)
        return TPT_ECUDA;
    p->launches_last = solve_launches + 2;
    return TPT_OK;
}

int tpt_plan_destroy(tpt_plan *p) {
    if (!p) return TPT_OK;
    cudaError_t e = cudaDeviceSynchronize();
    free_plan(p);
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

int tpt_plan_get_eigen(const tpt_plan *p, int dir, double *lambda_host, double *qtilde_host) {
    if (!p || (dir != 0 && dir != 1)) return TPT_EINVAL;
    const std::vector<double> &l = dir == 0 ? p->lamx : p->lamy;
    const std::vector<double> &q = dir == 0 ? p->qx : p->qy;
    if (!(p->dirs & (1 << dir))) return TPT_EINVAL;   // this plan does not diagonalise that direction
    if (qtilde_host && q.empty()) return TPT_EINVAL;   // fast-transform direction: the basis is not stored (closed form, fft.cu)
    if (lambda_host) std::memcpy(lambda_host, l.data(), l.size() * sizeof(double));
    if (qtilde_host) std::memcpy(qtilde_host, q.data(), q.size() * sizeof(double));
    return TPT_OK;
}

int tpt_plan_is_singular(const tpt_plan *p) { return p ? p->singular : TPT_EINVAL; }

int tpt_host_eigen(int n, const double *faces, int bc, int base_kind, double *lambda_host, double *qtilde_host) {
    if (!tpt::faces_valid(n, faces) || !bc_valid(bc) || (bc == TPT_BC_PERIODIC && n < 3)) return TPT_EINVAL;
    if (base_kind != 0 && base_kind != 1) return TPT_EINVAL;
    try {
        tpt::Operator1D op;
        tpt::build_operator(n, faces, bc, op);
        std::vector<double> lam, q;
        if (tpt::eigen_decompose(op, lam, q, base_kind) != 0) return TPT_ENUMERIC;
        if (lambda_host) std::memcpy(lambda_host, lam.data(), lam.size() * sizeof(double));
        if (qtilde_host) std::memcpy(qtilde_host, q.data(), q.size() * sizeof(double));
    } catch (const std::bad_alloc &) {
        return TPT_ENOMEM;
    } catch (...) {
        return TPT_ENUMERIC;
    }
    return TPT_OK;
}

int tpt_debug_sweep_geometry(int nz, int blocked, int sharded, int *out12) {
    if (!out12 || (sharded && !blocked)) return TPT_EINVAL;
    return tpt::thomas_onchip_geometry(nz, blocked != 0, sharded != 0, out12) ? TPT_OK : TPT_EINVAL;
}

int tpt_debug_set_eigen_base(int base_kind) {
    if (base_kind != 0 && base_kind != 1) return TPT_EINVAL;
    g_eigen_base = base_kind;
    return TPT_OK;
}

int tpt_plan_device_bytes(const tpt_plan *p, size_t *bytes_out) {
    if (!p || !bytes_out) return TPT_EINVAL;
    size_t b = 2 * ((size_t)p->nx * p->nx + (size_t)p->ny * p->ny) * sizeof(double);
    b += ((size_t)p->nx + p->ny + 4 * (size_t)p->nz + 8) * sizeof(double);
    b += (2 * ((size_t)p->nx + p->ny + p->nz) + 16) * sizeof(double);                       // staggered-grid geometry
    if (p->d_abc) b += 16 * ((size_t)p->nz + tpt::THOMAS_TABLE_PAD) * sizeof(double);       // sweep tables (thomas_onchip_tables)
    for (int d = 0; d < 2; ++d)
        if (p->d_fft[d]) b += (size_t)8 * (d == 0 ? p->nx : p->ny) * sizeof(double);        // twiddle tables (upper bound)
    b += p->points() * sizeof(double) * ((size_t)p->work_fields + (p->d_stage ? 1 : 0));
    b += 2 * p->slab_elems * sizeof(double);                                                // slab pipeline buffers (lazy)
    if (p->cyclic) b += (p->points() + (size_t)p->nx * p->ny) * sizeof(double);             // periodic z: q field + per-column factors
    *bytes_out = b;
    return TPT_OK;
}

int tpt_stage(tpt_plan *p, int slot, const double *in_dev, double *out_dev, void *cuda_stream) {
    if (!p || !in_dev || !out_dev || slot < 0 || slot >= TPT_K_COUNT) return TPT_EINVAL;
    if (!aligned16(in_dev) || !aligned16(out_dev) || !on_plan_device(p)) return TPT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0;
    if (!slot_active(p, slot)) return TPT_EINVAL;   // this plan does not diagonalise that direction
    if (slot == TPT_K_THOMAS) return run_thomas(p, in_dev, out_dev, p->d_work, st, &launches);
    if (in_dev == out_dev) return TPT_EINVAL;   // the transforms are out of place
    return run_slot(p, slot, in_dev, out_dev, st, &launches, 0, p->nz);
}

int tpt_plan_set_profiling(tpt_plan *p, int enabled) {
    if (!p) return TPT_EINVAL;
    p->profiling = enabled ? 1 : 0;
    return TPT_OK;
}

int tpt_plan_get_kernel_times(tpt_plan *p, float *ms_host, int *launches_out, int *solves_out) {
    if (!p || !ms_host) return TPT_EINVAL;
    const size_t per = TPT_K_COUNT + 1;
    const size_t solves = p->ev_used / per;
    if (solves == 0) return TPT_EINVAL;
    if (cudaEventSynchronize(p->ev_pool[p->ev_used - 1]) != cudaSuccess) return TPT_ECUDA;
    double sum[TPT_K_COUNT] = {0, 0, 0, 0, 0};
    for (size_t q = 0; q < solves; ++q)
        for (int s = 0; s < TPT_K_COUNT; ++s) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, p->ev_pool[q * per + s], p->ev_pool[q * per + s + 1]) != cudaSuccess)
                return TPT_ECUDA;
            sum[s] += ms;
        }
    for (int s = 0; s < TPT_K_COUNT; ++s) ms_host[s] = (float)(sum[s] / (double)solves);
    if (launches_out) *launches_out = (int)p->launches_accum;
    if (solves_out) *solves_out = (int)solves;
    p->ev_used = 0;
    p->launches_accum = 0;
    return TPT_OK;
}

int tpt_plan_get_paths(const tpt_plan *p, int *paths_out) {
    if (!p || !paths_out) return TPT_EINVAL;
    const bool blk = use_blocked(p);
    const bool fused = use_fused_small(p);
    double *w = p->d_work;   // stands for any 16-byte aligned field
    for (int s = 0; s < TPT_K_COUNT; ++s) {
        int path = TPT_PATH_NONE;
        if (fused) {
            path = (s == TPT_K_THOMAS || slot_active(p, s)) ? TPT_PATH_FUSED_SMALL : TPT_PATH_NONE;
        } else if (s == TPT_K_THOMAS) {
            const bool onchip = p->thomas_variant == 1 && tpt::thomas_onchip_supported(p->nx, p->ny, p->nz);
            path = !onchip ? TPT_PATH_THOMAS_STREAM : (blk ? TPT_PATH_THOMAS_BLOCKED : TPT_PATH_THOMAS_ONCHIP);
        } else if (slot_active(p, s)) {
            const int d = (s == TPT_K_FWD_X || s == TPT_K_INV_X) ? 0 : 1;
            if (p->transform[d] == TPT_TRANSFORM_FFT) {
                path = TPT_PATH_FFT;
            } else {
                const tpt::GemmArgs g = d == 0 ? gemm_x(p, w, w, p->d_xfwd, 0, p->nz)
                                               : gemm_y(p, w, w, p->d_yfwd, 0, p->nz, blk && s == TPT_K_INV_Y, blk && s == TPT_K_FWD_Y);
                if (p->gemm_variant == 2 && tpt::gemm_tma_supported(g)) path = TPT_PATH_GEMM_TMA;
                else if (p->gemm_variant >= 1 && tpt::gemm_dmma_supported(g)) path = TPT_PATH_GEMM_CPASYNC;
                else path = TPT_PATH_GEMM_GENERIC;
            }
        }
        paths_out[s] = path;
    }
    return TPT_OK;
}

int tpt_plan_set_gemm_variant(tpt_plan *p, int variant) {
    if (!p || variant < 0 || variant > 2) return TPT_EINVAL;
    p->gemm_variant = variant;
    return TPT_OK;
}

int tpt_plan_set_slab_groups(tpt_plan *p, int groups) {
    if (!p || groups < -1) return TPT_EINVAL;
    p->slab_groups = groups;
    return TPT_OK;
}

int tpt_plan_launches(const tpt_plan *p) { return p ? p->launches_last : TPT_EINVAL; }

int tpt_plan_set_fused_small(tpt_plan *p, int enabled) {
    if (!p) return TPT_EINVAL;
    p->fused_small = enabled ? 1 : 0;
    return TPT_OK;
}

int tpt_plan_set_thomas_variant(tpt_plan *p, int variant) {
    if (!p || (variant != 0 && variant != 1)) return TPT_EINVAL;
    p->thomas_variant = variant;
    return TPT_OK;
}

int tpt_fill_uniform(double *out_dev, size_t count, unsigned long long seed, unsigned long long offset, void *cuda_stream) {
    if ((!out_dev && count) || !aligned8(out_dev)) return TPT_EINVAL;
    cudaError_t e = tpt::launch_fill_uniform(out_dev, count, seed, offset, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
    return TPT_OK;
}

int tpt_fp64_peak(int kind, double *tflops_out) {
    if (!tflops_out || (kind != 0 && kind != 1)) return TPT_EINVAL;
    cudaError_t e = tpt::run_fp64_peak(kind, tflops_out);
    if (e != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
    return TPT_OK;
}

const char *tpt_strerror(int status) {
    switch (status) {
        case TPT_OK: return "ok";
        case TPT_EINVAL: return "invalid argument";
        case TPT_ENOMEM: return "out of memory";
        case TPT_ECUDA: return "CUDA error (no sm_100 device, or a runtime/launch failure)";
        case TPT_ENUMERIC: return "plan-time eigen-decomposition missed its accuracy rule";
        case TPT_ELIMIT: return "grid larger than the fixed capacity of a no-allocation entry point (TPT_STATIC_SCRATCH_POINTS)";
        default: return "unknown status";
    }
}

const char *tpt_version(void) { return "tpt 0.1 (sm_100a)"; }

}  // extern "C"
