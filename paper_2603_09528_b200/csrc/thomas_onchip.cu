// thomas_onchip.cu — step 2.3 (Eq. 11 at PAPER.md:161–163) with the whole z-column resident on chip:
// every point of the field is read from HBM once and written once (16 B/pt, the algorithmic minimum).
//
// A CTA owns tiles of 16 neighbouring (kx,ky) columns x nz rows, staged in shared memory by 2-D tiled TMA
// (boxes of 16 columns x up to 256 rows; 128-byte rows) through an NBUF-deep ring, so the load of the next tile
// and the store of the previous one overlap the arithmetic of the current one (persistent CTAs).
// (Row-by-row 1-D bulk copies were measured first: the TMA unit then sustains only ~1 copy / 17 cycles per SM,
// 2.2 TB/s chip-wide — hence the tensor map.)
//
// Inside a tile each column is cut into S segments of M rows, one thread per (column, segment):
//   1. cold forward elimination of the segment (Thomas forward sweep started as if the segment's first
//      row had no lower neighbour), carrying the fill-in column g_t that multiplies x_l, the last unknown
//      of the previous segment:          x_t + c'_t x_{t+1} + g_t x_l = d_t
//      and, in the same loop, the first row expressed through the segment's own last unknown:
//                                        x_first = DD - GG x_l + PI x_last
//   2. the S last unknowns of a column satisfy a tridiagonal system (Schur complement of the segment
//      interiors); it is solved by parallel cyclic reduction among the S threads of the column;
//   3. back substitution inside the segment:  x_t = d_t - g_t x_l - c'_t x_{t+1}.
// This is the Thomas elimination re-associated (exact in exact arithmetic; the matrix is diagonally
// dominant so no pivoting is needed, A13).  c'_t and g_t stay in registers, d_t / x_t in the tile.
#include <cuda.h>

#include <vector>

#include "kernels.cuh"
#include "ptx.cuh"

namespace tpt {

namespace {

constexpr int TCOLS = 16;                       // columns per tile: one 128-byte row per z level
constexpr int ROW_BYTES = TCOLS * (int)sizeof(double);

template <int M, int MAXT>
__global__ void __launch_bounds__(MAXT)
thomas_onchip_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_out,
                     const double *__restrict__ tab_reg,
                     const double *__restrict__ tab_null, const double *__restrict__ lamx,
                     const double *__restrict__ lamy, int nx, int nz, int S, int nbuf, int box_rows, int nbox,
                     int buf_rows, double shift0, int singular, int ntiles) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const size_t tile_elems = (size_t)buf_rows * TCOLS;             // buf_rows = max(S*M, nbox*box_rows) >= nz
    double *bufs = reinterpret_cast<double *>(smem_raw);            // nbuf x tile_elems
    double *scratch = bufs + (size_t)nbuf * tile_elems;             // 2 sets x 3 x S x 16
    uint64_t *full = reinterpret_cast<uint64_t *>(scratch + 6 * S * TCOLS);

    const int tid = threadIdx.x;
    const int col = tid & (TCOLS - 1);
    const int seg = tid >> 4;

    if (tid == 0) {
        ptx::tma_prefetch_desc(&tmap);
        ptx::tma_prefetch_desc(&tmap_out);
        for (int b = 0; b < nbuf; ++b) ptx::mbar_init(&full[b], 1);
        ptx::fence_mbar_init();
    }
    // rows the TMA boxes never reach (past nbox*box_rows) must read as zero: identity rows with p = 0
    for (int b = 0; b < nbuf; ++b)
        for (int e = nbox * box_rows * TCOLS + tid; e < (int)tile_elems; e += blockDim.x)
            bufs[(size_t)b * tile_elems + e] = 0.0;
    __syncthreads();

    auto issue_load = [&](int tile, int b) {      // one thread: nbox boxes of box_rows x 16 doubles
        if (tid != 0) return;
        ptx::mbar_arrive_expect_tx(&full[b], (uint32_t)((size_t)nbox * box_rows * ROW_BYTES));
        double *dst = bufs + (size_t)b * tile_elems;
        for (int q = 0; q < nbox; ++q)
            ptx::tma_load_2d(dst + (size_t)q * box_rows * TCOLS, &tmap, tile * TCOLS, q * box_rows, &full[b]);
    };

    const int first = blockIdx.x;
    const int n_my = first < ntiles ? (ntiles - first + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    for (int p = 0; p < nbuf - 1 && p < n_my; ++p) issue_load(first + p * (int)gridDim.x, p);

    const int k0 = seg * M;
    const int me = seg * TCOLS + col;
    const int STR = S * TCOLS;
    double *const set0 = scratch, *const set1 = scratch + 3 * STR;
    int b = 0;
    uint32_t parity = 0;
    for (int it = 0; it < n_my; ++it) {
        const int tile = first + it * (int)gridDim.x;
        double *buf = bufs + (size_t)b * tile_elems + (size_t)k0 * TCOLS + col;   // my segment, my column
        const int gcol = tile * TCOLS + col;
        const double s = __ldg(lamx + gcol % nx) + __ldg(lamy + gcol / nx) + shift0;
        // the null column of a singular plan reads a table whose last row is "-x = p", and zeroes p
        const bool null_col = singular && gcol == 0;
        const double2 *tab = reinterpret_cast<const double2 *>(null_col ? tab_null : tab_reg) + 2 * k0;

        ptx::bulk_wait_read<0>();              // (thread 0) the previous tile's store has left shared memory
        ptx::mbar_wait(&full[b], parity);
        if (null_col && (nz - 1) / M == seg) buf[((nz - 1) - k0) * TCOLS] = 0.0;

        // ---- 1. cold forward elimination of rows k0 .. k0+M-1 ------------------------------------
        double cp[M], g[M];
        double pi = 1.0, DD = 0.0, GG = 0.0, dprev = 0.0, rprev = 0.0;
#pragma unroll
        for (int t = 0; t < M; ++t) {
            const double2 t0 = __ldg(tab + 2 * t);         // { a_k c_{k-1}, b_k }
            const double2 t1 = __ldg(tab + 2 * t + 1);     // { a_k, c_k }
            const double p = buf[t * TCOLS];
            const double bb = t0.y + s;
            const double den = t == 0 ? bb : fma(-t0.x, rprev, bb);
            const double r = ptx::fast_rcp(den);
            cp[t] = t1.y * r;
            const double d = (t == 0 ? p : fma(-t1.x, dprev, p)) * r;
            g[t] = (t == 0 ? t1.x : -t1.x * g[t - 1]) * r;
            buf[t * TCOLS] = d;
            if (t < M - 1) {
                DD = fma(pi, d, DD);
                GG = fma(pi, g[t], GG);
                pi = -pi * cp[t];
            }
            dprev = d;
            rprev = r;
        }
        // ---- 2. reduced system for the last unknown X of each segment ------------------------------
        //   g_last X_{s-1} + (1 - c'_last GG_{s+1}) X_s + (c'_last PI_{s+1}) X_{s+1} = d_last - c'_last DD_{s+1}
        set0[me] = DD;
        set0[STR + me] = GG;
        set0[2 * STR + me] = pi;
        __syncthreads();
        // thread 0 has passed bulk_wait_read: the ring slot stored from in the previous iteration is free
        if (it + nbuf - 1 < n_my) {
            int nb = b + nbuf - 1;
            if (nb >= nbuf) nb -= nbuf;
            issue_load(first + (it + nbuf - 1) * (int)gridDim.x, nb);
        }
        double A = g[M - 1], C = 0.0, D = dprev;
        {
            double Bd = 1.0;
            if (seg + 1 < S) {
                const double cl = cp[M - 1];
                const int nb_ = me + TCOLS;
                Bd = fma(-cl, set0[STR + nb_], 1.0);
                C = cl * set0[2 * STR + nb_];
                D = fma(-cl, set0[nb_], D);
            }
            const double rB = ptx::fast_rcp(Bd);
            A *= rB;
            C *= rB;
            D *= rB;
        }
        // parallel cyclic reduction on  X_s + A X_{s-d} + C X_{s+d} = D
        double *wr = set1, *rd = set0;
        for (int dlt = 1; dlt < S; dlt <<= 1) {
            wr[me] = A;
            wr[STR + me] = C;
            wr[2 * STR + me] = D;
            __syncthreads();
            double Al = 0.0, Cl = 0.0, Dl = 0.0, Ah = 0.0, Ch = 0.0, Dh = 0.0;
            if (seg - dlt >= 0) {
                const int o = me - dlt * TCOLS;
                Al = wr[o];
                Cl = wr[STR + o];
                Dl = wr[2 * STR + o];
            }
            if (seg + dlt < S) {
                const int o = me + dlt * TCOLS;
                Ah = wr[o];
                Ch = wr[STR + o];
                Dh = wr[2 * STR + o];
            }
            const double rB = ptx::fast_rcp(fma(-C, Ah, fma(-A, Cl, 1.0)));
            D = fma(-C, Dh, fma(-A, Dl, D)) * rB;
            A = -A * Al * rB;
            C = -C * Ch * rB;
            double *tmp = wr;
            wr = rd;
            rd = tmp;
        }
        wr[me] = D;                            // X_s
        __syncthreads();
        const double xl = seg > 0 ? wr[me - TCOLS] : 0.0;
        // ---- 3. back substitution -------------------------------------------------------------------
        double xk = D;
        buf[(M - 1) * TCOLS] = xk;
#pragma unroll
        for (int t = M - 2; t >= 0; --t) {
            xk = fma(-cp[t], xk, fma(-g[t], xl, buf[t * TCOLS]));
            buf[t * TCOLS] = xk;
        }
        ptx::fence_proxy_async();
        __syncthreads();
        if (tid == 0) {                        // rows past nz are clipped by the tensor map
            const double *src = bufs + (size_t)b * tile_elems;
            for (int q = 0; q < nbox; ++q)
                ptx::tma_store_2d(&tmap_out, tile * TCOLS, q * box_rows, src + (size_t)q * box_rows * TCOLS);
            ptx::bulk_commit();
        }
        if (++b == nbuf) {
            b = 0;
            parity ^= 1;
        }
    }
    ptx::bulk_wait<0>();
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libcuda is not linked directly).
using EncodeTiledFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                   const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(ptr);
    }
    return fn;
}

// field viewed as a 2-D tensor: dim0 = nx*ny contiguous columns, dim1 = nz rows of stride nx*ny
bool make_field_map(CUtensorMap *map, const double *x, size_t plane, int nz, int box_rows) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const cuuint64_t dims[2] = {(cuuint64_t)plane, (cuuint64_t)nz};
    const cuuint64_t strides[1] = {(cuuint64_t)plane * sizeof(double)};
    const cuuint32_t box[2] = {(cuuint32_t)TCOLS, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double *>(x), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int M, int MAXT>
cudaError_t launch_m(const double *in, double *x, const double *tab, const double *lamx, const double *lamy, int nx, int ny, int nz,
                     double shift0, int singular, int sms, cudaStream_t stream) {
    int S = (nz + M - 1) / M;
    if (S & 1) ++S;                                          // whole warps: 2 segments x 16 columns
    const int nbox = (nz + 255) / 256;                       // TMA boxes are at most 256 rows tall
    const int box_rows = (nz + nbox - 1) / nbox;
    const int buf_rows = S * M > nbox * box_rows ? S * M : nbox * box_rows;
    const size_t tile_bytes = (size_t)buf_rows * ROW_BYTES;
    const size_t fixed = (size_t)6 * S * TCOLS * sizeof(double) + 64;
    int nbuf = (int)((220 * 1024 - fixed) / tile_bytes);
    if (nbuf > 3) nbuf = 3;
    if (nbuf < 2) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)nbuf * tile_bytes + fixed;
    static bool configured = false;
    static int per_sm_cache[2] = {0, 0};                     // {threads*2^20 + smem key, blocks per SM}
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(thomas_onchip_kernel<M, MAXT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             220 * 1024);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const int threads = TCOLS * S;
    if (threads > MAXT) return cudaErrorInvalidConfiguration;
    const int key = threads * 4096 + (int)(smem / 64);
    if (per_sm_cache[0] != key) {
        int per_sm = 0;
        cudaError_t e =
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, thomas_onchip_kernel<M, MAXT>, threads, smem);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorInvalidConfiguration;
        per_sm_cache[0] = key;
        per_sm_cache[1] = per_sm;
    }
    CUtensorMap tmap, tmap_out;
    if (!make_field_map(&tmap, in, (size_t)nx * ny, nz, box_rows)) return cudaErrorUnknown;
    if (!make_field_map(&tmap_out, x, (size_t)nx * ny, nz, box_rows)) return cudaErrorUnknown;
    const int ntiles = (int)(((size_t)nx * ny) / TCOLS);
    int grid = sms * per_sm_cache[1];
    if (grid > ntiles) grid = ntiles;
    thomas_onchip_kernel<M, MAXT><<<grid, threads, smem, stream>>>(
        tmap, tmap_out, tab, tab + 4 * ((size_t)nz + THOMAS_TABLE_PAD), lamx, lamy, nx, nz, S, nbuf, box_rows, nbox, buf_rows, shift0,
        singular, ntiles);
    return cudaGetLastError();
}

}  // namespace

bool thomas_onchip_supported(int nx, int ny, int nz) {
    return ((size_t)nx * ny) % TCOLS == 0 && nz >= 2 && nz <= 768;
}

cudaError_t launch_thomas_onchip(const double *in, double *x, const double *tab, const double *lamx, const double *lamy, int nx, int ny,
                                 int nz, double shift0, int singular, int sms, cudaStream_t stream) {
    if (!thomas_onchip_supported(nx, ny, nz)) return cudaErrorInvalidValue;
    if (nz <= 128) return launch_m<8, 256>(in, x, tab, lamx, lamy, nx, ny, nz, shift0, singular, sms, stream);
    if (nz <= 512) return launch_m<16, 512>(in, x, tab, lamx, lamy, nx, ny, nz, shift0, singular, sms, stream);
    return launch_m<32, 384>(in, x, tab, lamx, lamy, nx, ny, nz, shift0, singular, sms, stream);
}

// Host side of the coefficient tables: rows [a_k c_{k-1}, b_k, a_k, c_k], padded with decoupled rows
// [0, -1, 0, 0] (pivot -1 + s < 0 for every mode since s <= 0); the second table is the null column's, with the
// last equation replaced by "-x = p" (the kernel zeroes p there): PAPER.md:219.
void thomas_onchip_tables(int nz, const double *a, const double *b, const double *c, std::vector<double> &out) {
    const size_t rows = (size_t)nz + THOMAS_TABLE_PAD;
    out.assign(8 * rows, 0.0);
    for (int v = 0; v < 2; ++v) {
        double *t = out.data() + (size_t)v * 4 * rows;
        for (size_t k = 0; k < rows; ++k) t[4 * k + 1] = -1.0;
        for (int k = 0; k < nz; ++k) {
            t[4 * k] = k > 0 ? a[k] * c[k - 1] : 0.0;
            t[4 * k + 1] = b[k];
            t[4 * k + 2] = a[k];
            t[4 * k + 3] = c[k];
        }
        if (v == 1) {
            double *last = t + 4 * (size_t)(nz - 1);
            last[0] = 0.0; last[1] = -1.0; last[2] = 0.0; last[3] = 0.0;
        }
    }
}

}  // namespace tpt
