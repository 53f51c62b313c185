// fused_small.cu — the whole solve (steps 2.1–2.5, + the null-mode gauge of PAPER.md:219) in ONE
// launch for grids that fit on chip (BASELINE.json configs[0], 16^3; up to 16384 points).
//
// Five separate kernels cost five launch latencies (31 µs per 16^3 solve back to back) for microseconds of work.  Here one
// thread-block CLUSTER of C <= 8 CTAs holds the field in its shared memories:
//   * CTA c owns the z-planes [k0_c, k0_{c+1}).  The transforms act plane by plane (Eq. 10, 12), so steps 2.1 + 2.2 and
//     2.4 + 2.5 run back to back in shared memory with block-level barriers only;
//   * CTA c also owns a block of (kx, ky) columns for step 2.3 (Eq. 11).  The two changes of ownership go through the
//     plan's workspace in L2 (the field is at most 128 KB) and are ordered by two cluster barriers
//     (barrier.cluster arrive.release / wait.acquire) — the single-GPU miniature of the sharded solve (sharded.cu).
// The transforms are plain DFMA register tiles out of shared memory: at these sizes the solve is latency-bound, and the
// FP64 tensor path (same 128 flop/clk/SM peak as DFMA on sm_100) would buy nothing.
#include <cuda_runtime.h>

#include <mutex>

#include "devonce.hpp"
#include "kernels.cuh"

namespace tpt {

namespace {

constexpr int THREADS = 256;

struct FusedParams {
    const double *rhs;
    double *out;
    double *work;                       // the plan's workspace: mode-space field between the cluster barriers
    const double *xfwd, *xinv;          // [i][m], [m][i]   (plan.hpp)
    const double *yfwd, *yinv;          // [m][j], [j][m]
    const double *az, *bz, *cz, *wz, *lamx, *lamy;
    int nx, ny, nz;
    int dirs;                           // bit 0: x diagonalised, bit 1: y diagonalised
    int singular;
    double shift0;
    int planes_per_cta, cols_per_cta;   // ceil(nz / C), ceil(nx ny / C)
    int buf_elems;                      // doubles per shared-memory field buffer
};

__device__ __forceinline__ void cluster_sync_all() {
    __threadfence();                    // this CTA's global writes are performed before the barrier releases them
    asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r));
    return r;
}

// out[r][m] = sum_i in[r][i] mat[i][m]   for `rows` lines of length n (steps 2.1 / 2.5): T x T register tiles (T = 4, or
// 2 when 4 x 4 tiles would leave most threads idle).  FULL: rows and n are multiples of 4 (no edge predicates, 16-byte
// loads of the matrix row).
template <bool FULL, int T>
__device__ void mul_right_t(const double *__restrict__ in, double *__restrict__ out, const double *__restrict__ mat, int rows, int n) {
    const int tn = (n + T - 1) / T, tr = (rows + T - 1) / T;
    for (int w = threadIdx.x; w < tn * tr; w += THREADS) {
        const int m0 = (w % tn) * T, r0 = (w / tn) * T;
        double acc[T][T] = {};
#pragma unroll 4
        for (int i = 0; i < n; ++i) {
            double a[T], b[T];
            if (FULL) {
#pragma unroll
                for (int q = 0; q < T; q += 2) {
                    const double2 v = *reinterpret_cast<const double2 *>(mat + i * n + m0 + q);
                    b[q] = v.x; b[q + 1] = v.y;
                }
#pragma unroll
                for (int q = 0; q < T; ++q) a[q] = in[(r0 + q) * n + i];
            } else {
#pragma unroll
                for (int q = 0; q < T; ++q) {
                    a[q] = r0 + q < rows ? in[(r0 + q) * n + i] : 0.0;
                    b[q] = m0 + q < n ? mat[i * n + m0 + q] : 0.0;
                }
            }
#pragma unroll
            for (int q = 0; q < T; ++q)
#pragma unroll
                for (int s = 0; s < T; ++s) acc[q][s] = fma(a[q], b[s], acc[q][s]);
        }
#pragma unroll
        for (int q = 0; q < T; ++q) {
            if (FULL) {
#pragma unroll
                for (int s = 0; s < T; s += 2)
                    *reinterpret_cast<double2 *>(out + (r0 + q) * n + m0 + s) = make_double2(acc[q][s], acc[q][s + 1]);
            } else {
#pragma unroll
                for (int s = 0; s < T; ++s)
                    if (r0 + q < rows && m0 + s < n) out[(r0 + q) * n + m0 + s] = acc[q][s];
            }
        }
    }
}
template <bool FULL>
__device__ __forceinline__ void mul_right(const double *in, double *out, const double *mat, int rows, int n) {
    if (((n + 3) >> 2) * ((rows + 3) >> 2) >= THREADS) mul_right_t<FULL, 4>(in, out, mat, rows, n);
    else mul_right_t<FULL, 2>(in, out, mat, rows, n);
}

// out[k][m][i] = sum_j mat[m][j] in[k][j][i]   per plane k (steps 2.2 / 2.4, no transpose)
template <bool FULL, int T>
__device__ void mul_left_t(const double *__restrict__ in, double *__restrict__ out, const double *__restrict__ mat, int planes, int ny, int nx) {
    const int ti = (nx + T - 1) / T, tm = (ny + T - 1) / T;
    const int per = ti * tm;
    for (int w = threadIdx.x; w < per * planes; w += THREADS) {
        const int k = w / per, v = w - k * per;
        const int i0 = (v % ti) * T, m0 = (v / ti) * T;
        const double *src = in + k * ny * nx;
        double acc[T][T] = {};
#pragma unroll 4
        for (int j = 0; j < ny; ++j) {
            double a[T], b[T];
            if (FULL) {
#pragma unroll
                for (int q = 0; q < T; q += 2) {
                    const double2 u = *reinterpret_cast<const double2 *>(src + j * nx + i0 + q);
                    b[q] = u.x; b[q + 1] = u.y;
                }
#pragma unroll
                for (int q = 0; q < T; ++q) a[q] = mat[(m0 + q) * ny + j];
            } else {
#pragma unroll
                for (int q = 0; q < T; ++q) {
                    a[q] = m0 + q < ny ? mat[(m0 + q) * ny + j] : 0.0;
                    b[q] = i0 + q < nx ? src[j * nx + i0 + q] : 0.0;
                }
            }
#pragma unroll
            for (int q = 0; q < T; ++q)
#pragma unroll
                for (int s = 0; s < T; ++s) acc[q][s] = fma(a[q], b[s], acc[q][s]);
        }
        double *dst = out + k * ny * nx;
#pragma unroll
        for (int q = 0; q < T; ++q) {
            if (FULL) {
#pragma unroll
                for (int s = 0; s < T; s += 2)
                    *reinterpret_cast<double2 *>(dst + (m0 + q) * nx + i0 + s) = make_double2(acc[q][s], acc[q][s + 1]);
            } else {
#pragma unroll
                for (int s = 0; s < T; ++s)
                    if (m0 + q < ny && i0 + s < nx) dst[(m0 + q) * nx + i0 + s] = acc[q][s];
            }
        }
    }
}
template <bool FULL>
__device__ __forceinline__ void mul_left(const double *in, double *out, const double *mat, int planes, int ny, int nx) {
    if (((nx + 3) >> 2) * ((ny + 3) >> 2) * planes >= THREADS) mul_left_t<FULL, 4>(in, out, mat, planes, ny, nx);
    else mul_left_t<FULL, 2>(in, out, mat, planes, ny, nx);
}

// global <-> shared copies with every load of a thread in flight at once (the solve is latency-bound at these sizes)
template <bool CG>
__device__ __forceinline__ void copy_in(double *dst, const double *src, int n) {
    int e = threadIdx.x;
    for (; e + 3 * THREADS < n; e += 4 * THREADS) {
        double v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) v[q] = CG ? __ldcg(src + e + q * THREADS) : __ldg(src + e + q * THREADS);
#pragma unroll
        for (int q = 0; q < 4; ++q) dst[e + q * THREADS] = v[q];
    }
    for (; e < n; e += THREADS) dst[e] = CG ? __ldcg(src + e) : __ldg(src + e);
}

// FP64 reciprocal: MUFU seed and one cubically convergent step (finite, normal, non-zero x: the Thomas pivots of a
// diagonally dominant matrix)
__device__ __forceinline__ double rcp3(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;\n" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);
}

template <bool FULL>
__global__ void __launch_bounds__(THREADS, 1) fused_small_kernel(const FusedParams p) {
    extern __shared__ __align__(16) double smem[];
    double *A = smem, *B = smem + p.buf_elems;
    double *Mx = B + p.buf_elems, *My = Mx + p.nx * p.nx;
    double *tab = My + p.ny * p.ny;      // a_k, b_k, c_k of T_z: read once, used by every column of the CTA
    const int c = (int)cluster_ctarank();
    const int plane = p.nx * p.ny;
    const int k0 = min(c * p.planes_per_cta, p.nz), k1 = min(k0 + p.planes_per_cta, p.nz);
    const int nk = k1 - k0, npts = nk * plane;
    const bool use_x = p.dirs & 1, use_y = p.dirs & 2;

    // ---- steps 2.1, 2.2 on the own planes ----------------------------------------------------------------------
    copy_in<true>(A, p.rhs + (size_t)k0 * plane, npts);
    if (use_x) copy_in<false>(Mx, p.xfwd, p.nx * p.nx);
    if (use_y) copy_in<false>(My, p.yfwd, p.ny * p.ny);
    for (int k = threadIdx.x; k < p.nz; k += THREADS) {
        tab[3 * k] = __ldg(p.az + k);
        tab[3 * k + 1] = __ldg(p.bz + k);
        tab[3 * k + 2] = __ldg(p.cz + k);
    }
    __syncthreads();
    double *cur = A, *oth = B;
    if (use_x) {
        mul_right<FULL>(cur, oth, Mx, nk * p.ny, p.nx);
        __syncthreads();
        double *t = cur; cur = oth; oth = t;
    }
    if (use_y) {
        mul_left<FULL>(cur, oth, My, nk, p.ny, p.nx);
        __syncthreads();
        double *t = cur; cur = oth; oth = t;
    }
    for (int e = threadIdx.x; e < npts; e += THREADS) p.work[(size_t)k0 * plane + e] = cur[e];
    // the inverse matrices replace the forward ones (their latency hides under the barrier and the sweep)
    if (use_x) copy_in<false>(Mx, p.xinv, p.nx * p.nx);
    if (use_y) copy_in<false>(My, p.yinv, p.ny * p.ny);
    cluster_sync_all();

    // ---- step 2.3 on the own columns: Thomas, one thread per column, d' and c' in shared memory ------------------
    {
        const int c0 = min(c * p.cols_per_cta, plane), c1 = min(c0 + p.cols_per_cta, plane);
        const int nc = c1 - c0;
        double *dp = A, *cp = B;        // [k][column of this CTA]
        // the columns arrive with every load in flight at once (a per-thread walk down z would pay one L2 latency per row)
        {
            const int tot = p.nz * nc;
            int e = threadIdx.x;
            for (; e + 3 * THREADS < tot; e += 4 * THREADS) {
                double v[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int ee = e + q * THREADS, k = ee / nc;
                    v[q] = __ldcg(p.work + (size_t)k * plane + c0 + (ee - k * nc));
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) dp[e + q * THREADS] = v[q];
            }
            for (; e < tot; e += THREADS) {
                const int k = e / nc;
                dp[e] = __ldcg(p.work + (size_t)k * plane + c0 + (e - k * nc));
            }
        }
        __syncthreads();
        for (int t = threadIdx.x; t < nc; t += THREADS) {
            const int col = c0 + t;
            const double s = __ldg(p.lamx + col % p.nx) + __ldg(p.lamy + col / p.nx) + p.shift0;
            const bool null_col = p.singular && col == 0;
            double cprev = 0.0, dprev = 0.0;
#pragma unroll 4
            for (int k = 0; k < p.nz; ++k) {
                const double a = tab[3 * k];
                const double den = fma(-a, cprev, tab[3 * k + 1] + s);
                if (k == p.nz - 1 && null_col) {       // vanishing final pivot: modal unknown := 0
                    cprev = 0.0;
                    dprev = 0.0;
                } else {
                    const double r = rcp3(den);
                    cprev = tab[3 * k + 2] * r;
                    dprev = fma(-a, dprev, dp[k * nc + t]) * r;
                }
                cp[k * nc + t] = cprev;
                dp[k * nc + t] = dprev;
            }
            double xn = dprev, wsum = 0.0, wlen = 0.0;
#pragma unroll 4
            for (int k = p.nz - 1; k >= 0; --k) {
                if (k < p.nz - 1) xn = fma(-cp[k * nc + t], xn, dp[k * nc + t]);
                dp[k * nc + t] = xn;
                if (null_col) {
                    const double w = __ldg(p.wz + k);
                    wsum = fma(w, xn, wsum);
                    wlen += w;
                }
            }
            if (null_col) {     // gauge: zero dz-weighted mean of the null column (A7)
                const double mean = wsum / wlen;
                for (int k = 0; k < p.nz; ++k) dp[k * nc + t] -= mean;
            }
        }
        __syncthreads();
        for (int e = threadIdx.x; e < p.nz * nc; e += THREADS) {
            const int k = e / nc;
            p.work[(size_t)k * plane + c0 + (e - k * nc)] = dp[e];
        }
    }
    cluster_sync_all();

    // ---- steps 2.4, 2.5 on the own planes ----------------------------------------------------------------------
    copy_in<true>(A, p.work + (size_t)k0 * plane, npts);
    __syncthreads();
    cur = A;
    oth = B;
    if (use_y) {
        mul_left<FULL>(cur, oth, My, nk, p.ny, p.nx);
        __syncthreads();
        double *t = cur; cur = oth; oth = t;
    }
    if (use_x) {
        mul_right<FULL>(cur, oth, Mx, nk * p.ny, p.nx);
        __syncthreads();
        double *t = cur; cur = oth; oth = t;
    }
    for (int e = threadIdx.x; e < npts; e += THREADS) p.out[(size_t)k0 * plane + e] = cur[e];
}

constexpr size_t FUSED_MAX_POINTS = 16384;          // measured: 12 vs 31 us at 16^3, 23 vs 29 us at 24^3, 33 vs 29 us at 32^3
constexpr size_t FUSED_SMEM_MAX = 200 * 1024;

// cluster size: the largest of 8, 4, 2, 1 that leaves every CTA at least one plane
int cluster_size(int nz) { return nz >= 8 ? 8 : (nz >= 4 ? 4 : (nz >= 2 ? 2 : 1)); }

size_t fused_smem(int nx, int ny, int nz, int *buf_elems) {
    const int C = cluster_size(nz);
    const size_t plane = (size_t)nx * ny;
    const size_t ppc = (nz + C - 1) / C, cpc = (plane + C - 1) / C;
    size_t buf = ppc * plane > cpc * nz ? ppc * plane : cpc * (size_t)nz;
    buf = (buf + 1) & ~(size_t)1;
    if (buf_elems) *buf_elems = (int)buf;
    return (2 * buf + (size_t)nx * nx + (size_t)ny * ny + 3 * (size_t)nz) * sizeof(double);
}

}  // namespace

bool fused_small_supported(int nx, int ny, int nz) {
    if ((size_t)nx * ny * nz > FUSED_MAX_POINTS) return false;
    return fused_smem(nx, ny, nz, nullptr) <= FUSED_SMEM_MAX;
}

cudaError_t launch_fused_small(const FusedSmallArgs &a, cudaStream_t stream) {
    if (!fused_small_supported(a.nx, a.ny, a.nz)) return cudaErrorInvalidValue;
    FusedParams p{};
    p.rhs = a.rhs; p.out = a.out; p.work = a.work;
    p.xfwd = a.xfwd; p.xinv = a.xinv; p.yfwd = a.yfwd; p.yinv = a.yinv;
    p.az = a.az; p.bz = a.bz; p.cz = a.cz; p.wz = a.wz; p.lamx = a.lamx; p.lamy = a.lamy;
    p.nx = a.nx; p.ny = a.ny; p.nz = a.nz;
    p.dirs = a.dirs; p.singular = a.singular; p.shift0 = a.shift0;
    const int C = cluster_size(a.nz);
    p.planes_per_cta = (a.nz + C - 1) / C;
    p.cols_per_cta = (a.nx * a.ny + C - 1) / C;
    const size_t smem = fused_smem(a.nx, a.ny, a.nz, &p.buf_elems);
    static DeviceOnce configured;
    cudaError_t e = configured.run([&] {
        cudaError_t q = cudaFuncSetAttribute(fused_small_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSED_SMEM_MAX);
        if (q == cudaSuccess) q = cudaFuncSetAttribute(fused_small_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSED_SMEM_MAX);
        return q;
    });
    if (e != cudaSuccess) return e;
    // 16-byte register-tile loads need whole 4-element groups and 16-byte aligned rows in every shared-memory array
    const bool full = a.nx % 4 == 0 && a.ny % 4 == 0;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(C);
    cfg.blockDim = dim3(THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return full ? cudaLaunchKernelEx(&cfg, fused_small_kernel<true>, p) : cudaLaunchKernelEx(&cfg, fused_small_kernel<false>, p);
}

// ---- the same launch with its mode-space scratch in a static device array (tpt_solve_static_scratch, tpt.h) ---------
// For callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): nothing on
// this call path calls cudaMalloc, cudaFree or an allocating library routine.  Every GPU that loads the library holds
// the array (STATIC_SCRATCH_POINTS * 8 bytes = 128 KiB) until exit.  All calls on a device share it: calls that overlap
// on the GPU (two streams, two host threads) race on it.  It keeps the last call's contents, which is harmless here:
// every element the sweep reads was written by the same launch (each CTA stores its own z-planes before the first
// cluster barrier, together all nx ny nz points), so nothing has to start at zero.
static __device__ __align__(256) double static_scratch[STATIC_SCRATCH_POINTS];

cudaError_t launch_fused_small_static(const FusedSmallArgs &a, cudaStream_t stream) {
    if (a.nx < 1 || a.ny < 1 || a.nz < 1 || (size_t)a.nx * a.ny * a.nz > STATIC_SCRATCH_POINTS) return cudaErrorInvalidValue;
    // In host code `static_scratch` is a host-side stand-in, not a device address: the address a kernel may use comes from
    // cudaGetSymbolAddress, per device (every device has its own instance), with that device current.
    static std::mutex m;
    static double *addr[64] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    double *ptr = nullptr;
    {
        std::lock_guard<std::mutex> lock(m);
        if (dev >= 0 && dev < 64) ptr = addr[dev];
        if (!ptr) {
            e = cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), static_scratch);
            if (e != cudaSuccess) return e;
            if (!ptr) return cudaErrorInvalidSymbol;
            if (dev >= 0 && dev < 64) addr[dev] = ptr;
        }
    }
    FusedSmallArgs b = a;
    b.work = ptr;
    return launch_fused_small(b, stream);
}

}  // namespace tpt
