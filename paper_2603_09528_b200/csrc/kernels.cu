// kernels.cu — hand-written sm_100a kernels of the tensor-product–Thomas solve (steps 2.1–2.5,
// PAPER.md:181–185).  FP64 throughout.
//
//   gemm_dmma_kernel     eigenbasis transforms (steps 2.1, 2.2, 2.4, 2.5) as row-major batched GEMMs
//                        on the FP64 tensor path (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4, the native
//                        FP64 MMA shape of sm_100a), cp.async multi-stage shared-memory pipeline.
//   gemm_generic_kernel  same contraction with plain DFMA tiles for shapes the DMMA kernel does not
//                        take (tiny / ragged grids).
//   thomas_kernel        step 2.3: one thread per (kx,ky) column, coalesced along x.
//   gauge_kernel         null-mode gauge of a singular plan (A7).
#include "kernels.cuh"
#include "ptx.cuh"

namespace tpt {

using ptx::cp_async16;
using ptx::cp_async_commit;
using ptx::cp_async_wait;
using ptx::dmma884;

// ------------------------------------------------------------------------------------------------
// DMMA GEMM.  CTA tile BM x BN, k-slab BK = 16, warp tile WM x WN made of (WM/8) x (WN/8) m8n8k4 tiles.
// Shared memory per stage: A tile [BM][BK+4] and B tile [BK][BN+4] doubles; the +4 padding makes
// both fragment loads (8-byte, half-warp wavefronts) bank-conflict free.
// Requirements (checked by gemm_dmma_supported): M % BM == 0, N % BN == 0, K % 16 == 0, leading
// dimensions and batch strides even, base pointers 16-byte aligned.
// ------------------------------------------------------------------------------------------------
template <int BM, int BN, int WM, int WN, int STAGES>
struct DmmaCfg {
    static constexpr int BK = 16;
    static constexpr int APITCH = BK + 4;
    static constexpr int BPITCH = BN + 4;
    static constexpr int WARPS_M = BM / WM;
    static constexpr int WARPS_N = BN / WN;
    static constexpr int THREADS = WARPS_M * WARPS_N * 32;
    static constexpr int A_STAGE = BM * APITCH;
    static constexpr int B_STAGE = BK * BPITCH;
    static constexpr size_t SMEM_BYTES = (size_t)STAGES * (A_STAGE + B_STAGE) * sizeof(double);
};

template <int BM, int BN, int WM, int WN, int STAGES>
__global__ void __launch_bounds__(DmmaCfg<BM, BN, WM, WN, STAGES>::THREADS)
gemm_dmma_kernel(const double *__restrict__ A, const double *__restrict__ B, double *__restrict__ C,
                 int K, int64_t lda, int64_t ldb, int64_t ldc, int64_t strideA, int64_t strideB, int64_t strideC) {
    using Cfg = DmmaCfg<BM, BN, WM, WN, STAGES>;
    constexpr int BK = Cfg::BK, APITCH = Cfg::APITCH, BPITCH = Cfg::BPITCH, THREADS = Cfg::THREADS;
    constexpr int MT = WM / 8, NT = WN / 8;
    extern __shared__ __align__(16) double smem[];
    double *sA = smem;
    double *sB = smem + STAGES * Cfg::A_STAGE;

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, t = lane & 3;
    const int wm0 = (warp / Cfg::WARPS_N) * WM;
    const int wn0 = (warp % Cfg::WARPS_N) * WN;
    const int64_t m0 = (int64_t)blockIdx.y * BM;
    const int64_t n0 = (int64_t)blockIdx.x * BN;
    const int64_t batch = blockIdx.z;
    const double *Ag = A + batch * strideA + m0 * lda;
    const double *Bg = B + batch * strideB + n0;
    double *Cg = C + batch * strideC + m0 * ldc + n0;

    auto load_stage = [&](int stage, int kt) {
        double *a_dst = sA + stage * Cfg::A_STAGE;
        double *b_dst = sB + stage * Cfg::B_STAGE;
        const double *a_src = Ag + (int64_t)kt * BK;
        const double *b_src = Bg + (int64_t)kt * BK * ldb;
        constexpr int A_CHUNKS = BM * (BK / 2);          // 16-byte chunks
#pragma unroll
        for (int c = tid; c < A_CHUNKS; c += THREADS) {
            const int row = c >> 3, ch = c & 7;
            cp_async16(a_dst + row * APITCH + ch * 2, a_src + row * lda + ch * 2);
        }
        constexpr int B_ROW_CHUNKS = BN / 2;
        constexpr int B_CHUNKS = BK * B_ROW_CHUNKS;
#pragma unroll
        for (int c = tid; c < B_CHUNKS; c += THREADS) {
            const int row = c / B_ROW_CHUNKS, ch = c % B_ROW_CHUNKS;
            cp_async16(b_dst + row * BPITCH + ch * 2, b_src + row * ldb + ch * 2);
        }
    };

    double acc[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int KT = K / BK;
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < KT) load_stage(s, s);
        cp_async_commit();
    }
    for (int kt = 0; kt < KT; ++kt) {
        cp_async_wait<STAGES - 2>();   // k-slab kt has landed (for this thread's copies)
        __syncthreads();               // ... and for everyone's; also: slab kt-1 is no longer being read
        {
            const int nk = kt + STAGES - 1;
            if (nk < KT) load_stage(nk % STAGES, nk);
            cp_async_commit();
        }
        const double *a_s = sA + (kt % STAGES) * Cfg::A_STAGE + (wm0 + g) * APITCH + t;
        const double *b_s = sB + (kt % STAGES) * Cfg::B_STAGE + t * BPITCH + wn0 + g;
#pragma unroll
        for (int kk = 0; kk < BK / 4; ++kk) {
            double af[MT], bf[NT];
#pragma unroll
            for (int i = 0; i < MT; ++i) af[i] = a_s[i * 8 * APITCH + kk * 4];
#pragma unroll
            for (int j = 0; j < NT; ++j) bf[j] = b_s[kk * 4 * BPITCH + j * 8];
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cp_async_wait<0>();
    // epilogue: each lane owns C[g][2t..2t+1] of every 8x8 tile -> 16-byte stores
#pragma unroll
    for (int i = 0; i < MT; ++i) {
        double *crow = Cg + (int64_t)(wm0 + i * 8 + g) * ldc + wn0 + 2 * t;
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            double2 v = make_double2(acc[i][j][0], acc[i][j][1]);
            *reinterpret_cast<double2 *>(crow + j * 8) = v;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Generic DFMA GEMM: 64x64 CTA tile, 256 threads, each thread a 4x4 micro-tile strided by 16
// (rows ty+16r, cols tx+16c).  Any M, N, K; zero-filled edges.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
gemm_generic_kernel(const double *__restrict__ A, const double *__restrict__ B, double *__restrict__ C,
                    int M, int N, int K, int64_t lda, int64_t ldb, int64_t ldc,
                    int64_t strideA, int64_t strideB, int64_t strideC) {
    constexpr int TS = 64, BK = 16;
    __shared__ double As[TS][BK + 1];
    __shared__ double Bs[BK][TS];
    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const int64_t m0 = (int64_t)blockIdx.y * TS, n0 = (int64_t)blockIdx.x * TS;
    const int64_t batch = blockIdx.z;
    const double *Ab = A + batch * strideA;
    const double *Bb = B + batch * strideB;
    double *Cb = C + batch * strideC;
    double acc[4][4];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[r][c] = 0.0;
    for (int k0 = 0; k0 < K; k0 += BK) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int e = tid + 256 * q;
            const int row = e / BK, kk = e % BK;
            const int64_t gm = m0 + row;
            const int gk = k0 + kk;
            As[row][kk] = (gm < M && gk < K) ? Ab[gm * lda + gk] : 0.0;
            const int brow = e / TS, bcol = e % TS;
            const int gk2 = k0 + brow;
            const int64_t gn = n0 + bcol;
            Bs[brow][bcol] = (gk2 < K && gn < N) ? Bb[(int64_t)gk2 * ldb + gn] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < BK; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) a[r] = As[ty + 16 * r][kk];
#pragma unroll
            for (int c = 0; c < 4; ++c) b[c] = Bs[kk][tx + 16 * c];
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[r][c] = fma(a[r], b[c], acc[r][c]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int64_t gm = m0 + ty + 16 * r;
        if (gm >= M) continue;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int64_t gn = n0 + tx + 16 * c;
            if (gn < N) Cb[gm * ldc + gn] = acc[r][c];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// launch glue
// ------------------------------------------------------------------------------------------------
using CfgBig = DmmaCfg<128, 128, 32, 32, 3>;      // 16 warps, 3 stages (109.5 KB)
using CfgSmall = DmmaCfg<64, 64, 32, 32, 4>;      // 4 warps, 4 stages, for narrow problems

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static bool dmma_shape_ok(const GemmArgs &g, int bm, int bn) {
    return g.M % bm == 0 && g.N % bn == 0 && g.K % 16 == 0 && g.K >= 16 && (g.lda % 2) == 0 && (g.ldb % 2) == 0 &&
           (g.ldc % 2) == 0 && (g.strideA % 2) == 0 && (g.strideB % 2) == 0 && (g.strideC % 2) == 0 &&
           aligned16(g.A) && aligned16(g.B) && aligned16(g.C) && g.batch <= 65535 && g.M / bm <= 65535;
}

bool gemm_dmma_supported(const GemmArgs &g) { return dmma_shape_ok(g, 64, 64); }

cudaError_t gemm_configure() {
    cudaError_t e = cudaFuncSetAttribute(gemm_dmma_kernel<128, 128, 32, 32, 3>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CfgBig::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(gemm_dmma_kernel<64, 64, 32, 32, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)CfgSmall::SMEM_BYTES);
}

cudaError_t launch_gemm(const GemmArgs &g, int variant, cudaStream_t stream) {
    if (g.M <= 0 || g.N <= 0 || g.K <= 0 || g.batch <= 0) return cudaErrorInvalidValue;
    if (variant == 1 && dmma_shape_ok(g, 128, 128)) {
        dim3 grid(g.N / 128, g.M / 128, g.batch);
        gemm_dmma_kernel<128, 128, 32, 32, 3><<<grid, CfgBig::THREADS, CfgBig::SMEM_BYTES, stream>>>(
            g.A, g.B, g.C, g.K, g.lda, g.ldb, g.ldc, g.strideA, g.strideB, g.strideC);
        return cudaGetLastError();
    }
    if (variant == 1 && dmma_shape_ok(g, 64, 64)) {
        dim3 grid(g.N / 64, g.M / 64, g.batch);
        gemm_dmma_kernel<64, 64, 32, 32, 4><<<grid, CfgSmall::THREADS, CfgSmall::SMEM_BYTES, stream>>>(
            g.A, g.B, g.C, g.K, g.lda, g.ldb, g.ldc, g.strideA, g.strideB, g.strideC);
        return cudaGetLastError();
    }
    const int64_t gy = ((int64_t)g.M + 63) / 64;
    if (gy > 65535 || g.batch > 65535) {
        // fold rows into more batches is not possible in general; split the launch along M
        const int rows_per = 65535 * 64;
        for (int64_t r0 = 0; r0 < g.M; r0 += rows_per) {
            GemmArgs h = g;
            h.A = g.A + r0 * g.lda;
            h.C = g.C + r0 * g.ldc;
            h.M = (int)((g.M - r0 < rows_per) ? (g.M - r0) : rows_per);
            if (h.batch > 65535) return cudaErrorInvalidValue;
            cudaError_t e = launch_gemm(h, variant, stream);
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    }
    dim3 grid((g.N + 63) / 64, (unsigned)gy, g.batch);
    gemm_generic_kernel<<<grid, 256, 0, stream>>>(g.A, g.B, g.C, g.M, g.N, g.K, g.lda, g.ldb, g.ldc, g.strideA,
                                                  g.strideB, g.strideC);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// z sweep.  Thomas algorithm, one thread per column; element k of column (j,i) at x[i + nx*j + k*nx*ny]
// so a warp reads 256 contiguous bytes per k.  Forward sweep overwrites x with d' and writes
// c' to `cprime`; the back substitution reads both.  Loads are issued U at a time before the
// dependent recurrence so that U rows per thread are in flight.
//   den_k = (b_k + s) - a_k c'_{k-1},  c'_k = c_k/den_k,  d'_k = (p_k - a_k d'_{k-1})/den_k
//   x_k  = d'_k - c'_k x_{k+1}
// ------------------------------------------------------------------------------------------------
template <int U>
__global__ void __launch_bounds__(128)
thomas_kernel(double *x, double *__restrict__ cprime, const double *__restrict__ az, const double *__restrict__ bz,
              const double *__restrict__ cz, const double *__restrict__ lamx, const double *__restrict__ lamy, int nx,
              int ny, int nz, double shift0, int singular, double b0_null) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    if (i >= nx) return;
    const size_t plane = (size_t)nx * ny;
    double *xc = x + (size_t)i + (size_t)nx * j;
    double *cc = cprime + (size_t)i + (size_t)nx * j;
    const double s = lamx[i] + lamy[j] + shift0;
    const bool null_col = singular && i == 0 && j == 0;

    double r = 1.0 / ((null_col ? b0_null : __ldg(bz)) + s);      // (cyclic sweep: the null column keeps the unmodified corner)
    double cprev = __ldg(cz) * r;
    double dprev = xc[0] * r;
    cc[0] = cprev;
    xc[0] = dprev;
    for (int k0 = 1; k0 < nz; k0 += U) {
        double v[U];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (k0 + u < nz) v[u] = xc[(size_t)(k0 + u) * plane];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int k = k0 + u;
            if (k < nz) {
                const double a = __ldg(az + k);
                const double den = (__ldg(bz + k) + s) - a * cprev;
                if (k == nz - 1 && null_col) {   // vanishing final pivot: modal unknown := 0
                    cprev = 0.0;
                    dprev = 0.0;
                } else {
                    r = 1.0 / den;
                    cprev = __ldg(cz + k) * r;
                    dprev = (v[u] - a * dprev) * r;
                }
                cc[(size_t)k * plane] = cprev;
                xc[(size_t)k * plane] = dprev;
            }
        }
    }
    double xn = dprev;
    for (int k0 = nz - 2; k0 >= 0; k0 -= U) {
        double dv[U], cv[U];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (k0 - u >= 0) {
                dv[u] = xc[(size_t)(k0 - u) * plane];
                cv[u] = cc[(size_t)(k0 - u) * plane];
            }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (k0 - u >= 0) {
                xn = dv[u] - cv[u] * xn;
                xc[(size_t)(k0 - u) * plane] = xn;
            }
    }
}

cudaError_t launch_thomas(double *x, double *cprime, const double *az, const double *bz, const double *cz,
                          const double *lamx, const double *lamy, int nx, int ny, int nz, double shift0, int singular,
                          double b0_null, cudaStream_t stream) {
    if (ny > 65535) return cudaErrorInvalidValue;
    dim3 grid((nx + 127) / 128, ny);
    thomas_kernel<8><<<grid, 128, 0, stream>>>(x, cprime, az, bz, cz, lamx, lamy, nx, ny, nz, shift0, singular, b0_null);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Periodic z ("cyclic corner entries"; A19): the cyclic column matrix is the tridiagonal A'
// the sweep kernels solve (corners b_0 - g, b_{n-1} - c_{n-1} a_0 / g, one g per plan) plus a rank-one term, so
//     x = y - q (y_0 + r y_{n-1}) / (1 + q_0 + r q_{n-1}),   A' y = p,  A' q = u = (g, 0, .., 0, c_{n-1}),  r = a_0 / g
// (Sherman-Morrison).  q depends on the column's spectral shift only, not on the right-hand side: it is swept once at
// plan time and kept (one field), with rden = 1 / (1 + q_0 + r q_{n-1}) per column (0 for the null column of a singular
// plan, which the sweep itself gauges).  Per solve: the ordinary sweep, then this correction (24 B/pt).  Natural layout.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) cyclic_rhs_kernel(double *u, size_t cols, int nz, double g, double cn) {
    const size_t col = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= cols) return;
    for (int k = 0; k < nz; ++k) u[(size_t)k * cols + col] = k == 0 ? g : (k == nz - 1 ? cn : 0.0);
}

__global__ void __launch_bounds__(256) cyclic_rden_kernel(const double *__restrict__ q, double *__restrict__ rden, size_t cols, int nz,
                                                          double r, int singular) {
    const size_t col = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= cols) return;
    const double den = 1.0 + q[col] + r * q[(size_t)(nz - 1) * cols + col];
    rden[col] = (singular && col == 0) ? 0.0 : 1.0 / den;
}

__global__ void __launch_bounds__(256) cyclic_correct_kernel(double *x, const double *__restrict__ q, const double *__restrict__ rden,
                                                             size_t cols, int nz, double r) {
    const size_t col = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= cols) return;
    const double fact = (x[col] + r * x[(size_t)(nz - 1) * cols + col]) * __ldg(rden + col);
#pragma unroll 4
    for (int k = 0; k < nz; ++k) {
        const size_t e = (size_t)k * cols + col;
        x[e] = fma(-fact, __ldg(q + e), x[e]);
    }
}

cudaError_t launch_cyclic_rhs(double *u, size_t cols, int nz, double g, double cn, cudaStream_t stream) {
    cyclic_rhs_kernel<<<(unsigned)((cols + 255) / 256), 256, 0, stream>>>(u, cols, nz, g, cn);
    return cudaGetLastError();
}
cudaError_t launch_cyclic_rden(const double *q, double *rden, size_t cols, int nz, double r, int singular, cudaStream_t stream) {
    cyclic_rden_kernel<<<(unsigned)((cols + 255) / 256), 256, 0, stream>>>(q, rden, cols, nz, r, singular);
    return cudaGetLastError();
}
cudaError_t launch_cyclic_correct(double *x, const double *q, const double *rden, size_t cols, int nz, double r, cudaStream_t stream) {
    cyclic_correct_kernel<<<(unsigned)((cols + 255) / 256), 256, 0, stream>>>(x, q, rden, cols, nz, r);
    return cudaGetLastError();
}

// Null-mode gauge: x[k*plane] -= sum_k wz[k] x[k*plane] / sum_k wz[k]   (column i = j = 0).
__global__ void __launch_bounds__(256) gauge_kernel(double *x, const double *__restrict__ wz, size_t plane, int nz) {
    __shared__ double red_s[256], red_l[256];
    double s = 0.0, l = 0.0;
    for (int k = threadIdx.x; k < nz; k += 256) {
        s += wz[k] * x[(size_t)k * plane];
        l += wz[k];
    }
    red_s[threadIdx.x] = s;
    red_l[threadIdx.x] = l;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (threadIdx.x < w) {
            red_s[threadIdx.x] += red_s[threadIdx.x + w];
            red_l[threadIdx.x] += red_l[threadIdx.x + w];
        }
        __syncthreads();
    }
    const double mean = red_s[0] / red_l[0];
    for (int k = threadIdx.x; k < nz; k += 256) x[(size_t)k * plane] -= mean;
}

cudaError_t launch_gauge(double *x, const double *wz, size_t stride, int nz, cudaStream_t stream) {
    gauge_kernel<<<1, 256, 0, stream>>>(x, wz, stride, nz);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Seeded white-noise input generator on the device (the same counter-based recipe as
// paper_2603_09528_b200/inputs.py, restated): element t = 2u - 1 with u the top 53 bits of the splitmix64
// finaliser of (offset + t + (seed + 1) * 0x9E3779B97F4A7C15).  No solver arithmetic.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fill_uniform_kernel(double *out, size_t count, unsigned long long base) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < count; t += stride) {
        unsigned long long z = base + t;
        z ^= z >> 30;
        z *= 0xBF58476D1CE4E5B9ull;
        z ^= z >> 27;
        z *= 0x94D049BB133111EBull;
        z ^= z >> 31;
        out[t] = (double)(z >> 11) * 0x1.0p-52 - 1.0;
    }
}

cudaError_t launch_fill_uniform(double *out, size_t count, unsigned long long seed, unsigned long long offset, cudaStream_t stream) {
    if (count == 0) return cudaSuccess;
    const unsigned long long base = (seed + 1ull) * 0x9E3779B97F4A7C15ull + offset;
    size_t blocks = (count + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    fill_uniform_kernel<<<(unsigned)blocks, 256, 0, stream>>>(out, count, base);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// FP64 pipe microbenchmarks (roofline denominators; MEASURED_PEAKS.json has no FP64 entry).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) peak_dfma_kernel(double *out, int iters, double x, double y) {
    double acc[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) acc[q] = (double)(threadIdx.x + q);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 16; ++q) acc[q] = fma(acc[q], x, y);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 16; ++q) s += acc[q];
    if (s == 1.2345e300) out[0] = s;
}

__global__ void __launch_bounds__(512) peak_dmma_kernel(double *out, int iters, double a, double b) {
    double c[16][2];
#pragma unroll
    for (int q = 0; q < 16; ++q) c[q][0] = c[q][1] = (double)(threadIdx.x + q);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 16; ++q) dmma884(c[q][0], c[q][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 16; ++q) s += c[q][0] + c[q][1];
    if (s == 1.2345e300) out[0] = s;
}

cudaError_t run_fp64_peak(int kind, double *tflops) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double *out = nullptr;
    e = cudaMalloc(&out, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 4, threads = 512;
    const int iters = kind == 0 ? 4096 : 1024;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0);
        if (kind == 0) peak_dfma_kernel<<<blocks, threads>>>(out, iters, 0.999999, 1e-9);
        else peak_dmma_kernel<<<blocks, threads>>>(out, iters, 0.999999, 1e-9);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double flops;
        if (kind == 0) flops = (double)blocks * threads * iters * 16.0 * 2.0;
        else flops = (double)blocks * (threads / 32) * iters * 16.0 * 512.0;
        const double tf = flops / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (e == cudaSuccess) e = cudaGetLastError();
    *tflops = best;
    return e;
}

}  // namespace tpt
