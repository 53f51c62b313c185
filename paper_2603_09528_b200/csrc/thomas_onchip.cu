// thomas_onchip.cu — step 2.3 (Eq. 11 at PAPER.md:161–163) with the whole z-column resident on chip:
// every point of the field is read from HBM once and written once (16 B/pt, the algorithmic minimum).
//
// A CTA owns tiles of 16 (or 8, or 4) neighbouring (kx,ky) columns x nz rows, staged in shared memory by tiled TMA
// (boxes of up to 256 rows of 128, 64 or 32 bytes) through an NBUF-deep ring, so the load of the next tile and the
// store of the previous one overlap the arithmetic of the current one (persistent CTAs).  The field may be in the
// natural layout (rows nx*ny apart) or in the tile-blocked mode-space layout of kernels.cuh, where a 16-column tile
// is one dense block of nz*128 bytes; the tensor map hides the difference.  Launch shapes: choose_shape.
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

#include <type_traits>
#include <vector>

#include "devonce.hpp"
#include "kernels.cuh"
#include "ptx.cuh"
#include "tmap.hpp"

namespace tpt {

namespace {

// Destination of the solution tiles.  Plain solve: one tensor map over the output field.  Sharded solve (sharded.cu;
// PAPER.md:197-207, Algorithm 1 step 6): rows [k0[r], k0[r+1]) of every tile belong to rank r, whose z-slab buffer
// (tile-blocked, peer-mapped over NVLink) they are stored into directly — the transpose back to z-slabs is this
// kernel's own TMA store, not a collective.
struct StoreOne { CUtensorMap map; };
struct StorePeers {
    CUtensorMap map[MAX_PEERS];   // rank r's slab buffer as [16-column group][tile of the group][local z][columns]
    int k0[MAX_PEERS + 1];        // z-slab boundaries (even numbers, so 8-column rows stay 128-byte aligned in shared memory)
    int npeers;
    int box_rows;                 // rows per store box
    int group0;                   // index of this rank's first 16-column group in the peers' (global) group numbering
};

// Coefficient tables: stored [group of 4 segments][t][segment] for the launch's partition (thomas_onchip_tables).  In row
// order a warp's two 16-byte loads per row touched one 128-byte line per segment: 36 M sectors per launch at 512^3, 40 %
// of the kernel's LSU data-pipe wavefronts — the busiest unit (76 %, ncu); now one or two lines per load.  TS: the
// regular table is also copied to shared memory once per CTA and read from there (where it fits beside the tile ring).
template <int M, int TCOLS, int MAXT, int MINB, bool SH, bool TS>
__global__ void __launch_bounds__(MAXT, MINB)
thomas_onchip_kernel(const __grid_constant__ CUtensorMap tmap,
                     const __grid_constant__ typename std::conditional<SH, StorePeers, StoreOne>::type dst,
                     const double *__restrict__ tab_reg,
                     const double *__restrict__ tab_null, const double *__restrict__ lamx,
                     const double *__restrict__ lamy, const double *__restrict__ wz, int nx, int nz, int S, int nbuf,
                     int box_rows, int nbox, int buf_rows, double shift0, int singular, int ntiles) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const size_t tile_elems = (size_t)buf_rows * TCOLS;             // buf_rows >= nbox*box_rows >= nz; PRED: may be < S*M
    constexpr bool PRED = MINB > 1;                                 // thomas_geometry: which shapes keep fewer than S*M rows
    double *bufs = reinterpret_cast<double *>(smem_raw);            // nbuf x tile_elems
    double *scratch = bufs + (size_t)nbuf * tile_elems;             // 2 sets x 3 x S x 16
    uint64_t *full = reinterpret_cast<uint64_t *>(scratch + 6 * S * TCOLS);
    double2 *stab = reinterpret_cast<double2 *>(reinterpret_cast<unsigned char *>(full) + 128);   // TS: 2 * S*M entries

    const int tid = threadIdx.x;
    constexpr int ROW_BYTES = TCOLS * (int)sizeof(double);
    constexpr int SUB = 16 / TCOLS;              // tiles per 16-column group
    const int col = tid & (TCOLS - 1);
    const int seg = tid / TCOLS;

    if (tid == 0) {
        ptx::tma_prefetch_desc(&tmap);
        if constexpr (SH) {
            for (int r = 0; r < dst.npeers; ++r) ptx::tma_prefetch_desc(&dst.map[r]);
        } else {
            ptx::tma_prefetch_desc(&dst.map);
        }
        for (int b = 0; b < nbuf; ++b) ptx::mbar_init(&full[b], 1);
        ptx::fence_mbar_init();
    }
    if constexpr (!PRED) {        // rows the TMA boxes never reach (past nbox*box_rows) read as zero: identity rows with p = 0
        for (int b = 0; b < nbuf; ++b)
            for (int e = nbox * box_rows * TCOLS + tid; e < (int)tile_elems; e += blockDim.x) bufs[(size_t)b * tile_elems + e] = 0.0;
    }
    if constexpr (TS) {           // plan data, not the previous kernel's output: copied before the dependency wait
        for (int e = tid; e < 2 * ((S + 3) & ~3) * M; e += blockDim.x) stab[e] = __ldg(reinterpret_cast<const double2 *>(tab_reg) + e);
    }
    ptx::pdl_launch_dependents();
    __syncthreads();
    ptx::pdl_wait();              // the tiles are the previous kernel's output

    auto issue_load = [&](int tile, int b) {      // one thread: nbox boxes of box_rows x 16 doubles
        if (tid != 0) return;
        ptx::mbar_arrive_expect_tx(&full[b], (uint32_t)((size_t)nbox * box_rows * ROW_BYTES));
        double *dst = bufs + (size_t)b * tile_elems;
        for (int q = 0; q < nbox; ++q)
            ptx::tma_load_4d(dst + (size_t)q * box_rows * TCOLS, &tmap, 0, q * box_rows, tile % SUB, tile / SUB, &full[b]);
    };

    const int first = blockIdx.x;
    const int n_my = first < ntiles ? (ntiles - first + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    for (int p = 0; p < nbuf - 1 && p < n_my; ++p) issue_load(first + p * (int)gridDim.x, p);

    const int k0 = seg * M;
    // rows of my segment that exist in the tile buffer; the rest of the S*M rows (past nbox*box_rows) are decoupled
    // identity rows of the padded table with p = 0: they read as zero and are never written
    const int live = PRED ? buf_rows - k0 : M;
    const int me = seg * TCOLS + col;
    const int STR = S * TCOLS;
    double *const set0 = scratch, *const set1 = scratch + 3 * STR;
    int b = 0;
    uint32_t parity = 0;
    // the spectral shift of my column in the next tile is fetched one tile ahead (its latency hides under the sweep)
    auto shift_of = [&](int tile) {
        const int gc = tile * TCOLS + col;
        return __ldg(lamx + gc % nx) + __ldg(lamy + gc / nx) + shift0;
    };
    double s_next = n_my > 0 ? shift_of(first) : 0.0;
    for (int it = 0; it < n_my; ++it) {
        const int tile = first + it * (int)gridDim.x;
        double *buf = bufs + (size_t)b * tile_elems + (size_t)k0 * TCOLS + col;   // my segment, my column
        const int gcol = tile * TCOLS + col;
        const double s = s_next;
        if (it + 1 < n_my) s_next = shift_of(tile + (int)gridDim.x);
        // the null column of a singular plan reads a table whose last row is "-x = p", and zeroes p
        const bool null_col = singular && gcol == 0;
        // Global tables of this launch's partition (thomas_onchip_tables), stored [group of 4 segments][t][segment of the
        // group]: row k0 + t of segment `seg` at (((seg / 4) M + t) 4 + seg % 4) 32 bytes.  The (4 or 8) segments of a warp
        // then read one or two 128-byte lines per load, not one line each, at compile-time offsets (128 t bytes).
        const int tab_off = 2 * (((seg >> 2) * M) * 4 + (seg & 3));
        const double2 *tab = reinterpret_cast<const double2 *>(null_col ? tab_null : tab_reg) + tab_off;
        // the tile that holds the null column reads the tables from global memory (block-uniform choice)
        const bool tab_in_smem = TS && !(singular && tile == 0);

        ptx::bulk_wait_read<0>();              // (thread 0) the previous tile's store has left shared memory
        ptx::mbar_wait(&full[b], parity);
        if (null_col && (nz - 1) / M == seg) buf[((nz - 1) - k0) * TCOLS] = 0.0;

        // ---- 1. cold forward elimination of rows k0 .. k0+M-1 ------------------------------------
        double cp[M], g[M];
        double pi = 1.0, DD = 0.0, GG = 0.0, dprev = 0.0, rprev = 0.0;
        auto forward = [&](const double2 *tb, auto load) {
#pragma unroll
            for (int t = 0; t < M; ++t) {
                const double2 t0 = load(tb + 8 * t);                // { a_k c_{k-1}, b_k }
                const double2 t1 = load(tb + 8 * t + 1);            // { a_k, c_k }
                const double p = t < live ? buf[t * TCOLS] : 0.0;
                const double bb = t0.y + s;
                const double den = t == 0 ? bb : fma(-t0.x, rprev, bb);
                const double r = ptx::fast_rcp3(den);
                cp[t] = t1.y * r;
                const double d = (t == 0 ? p : fma(-t1.x, dprev, p)) * r;
                g[t] = (t == 0 ? t1.x : -t1.x * g[t - 1]) * r;
                if (t < live) buf[t * TCOLS] = d;
                if (t < M - 1) {
                    DD = fma(pi, d, DD);
                    GG = fma(pi, g[t], GG);
                    pi = -pi * cp[t];
                }
                dprev = d;
                rprev = r;
            }
        };
        if (tab_in_smem) forward(stab + tab_off, [](const double2 *q) { return *q; });
        else forward(tab, [](const double2 *q) { return __ldg(q); });
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
            // Early exit: once every coupling of the tile is below 1e-30 the remaining rounds would change D by less
            // than 1e-30 |D_neighbour| — nothing in FP64.  (High modes decouple after one or two rounds: |c'| << 1.)
            if (!__syncthreads_or(fmax(fabs(A), fabs(C)) > 1e-30)) break;
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
        if (M - 1 < live) buf[(M - 1) * TCOLS] = xk;
#pragma unroll
        for (int t = M - 2; t >= 0; --t) {
            xk = fma(-cp[t], xk, fma(-g[t], xl, t < live ? buf[t * TCOLS] : 0.0));
            if (t < live) buf[t * TCOLS] = xk;
        }
        // ---- null-mode gauge (A7), fused: the tile that holds column (0,0) of a singular
        // plan subtracts the dz-weighted mean of that column before it leaves the chip (block-uniform branch)
        if (singular && tile == 0) {
            __syncthreads();
            double ps = 0.0, pl = 0.0;
            if (col == 0) {
#pragma unroll
                for (int t = 0; t < M; ++t)
                    if (k0 + t < nz) {
                        const double w = __ldg(wz + k0 + t);
                        ps = fma(w, buf[t * TCOLS], ps);
                        pl += w;
                    }
            }
            set0[me] = ps;
            set0[STR + me] = pl;
            __syncthreads();
            double sum = 0.0, len = 0.0;
            for (int q = 0; q < S; ++q) {
                sum += set0[q * TCOLS];
                len += set0[STR + q * TCOLS];
            }
            const double mean = sum / len;
            if (col == 0) {
#pragma unroll
                for (int t = 0; t < M; ++t)
                    if (k0 + t < nz) buf[t * TCOLS] -= mean;
            }
        }
        ptx::fence_proxy_async();
        __syncthreads();
        if (tid == 0) {                        // rows past nz are clipped by the tensor map
            const double *src = bufs + (size_t)b * tile_elems;
            if constexpr (SH) {
                for (int r = 0; r < dst.npeers; ++r)
                    for (int kk = dst.k0[r]; kk < dst.k0[r + 1]; kk += dst.box_rows)
                        ptx::tma_store_4d(&dst.map[r], 0, kk - dst.k0[r], tile % SUB, dst.group0 + tile / SUB, src + (size_t)kk * TCOLS);
            } else {
                for (int q = 0; q < nbox; ++q)
                    ptx::tma_store_4d(&dst.map, 0, q * box_rows, tile % SUB, tile / SUB, src + (size_t)q * box_rows * TCOLS);
            }
            ptx::bulk_commit();
        }
        if (++b == nbuf) {
            b = 0;
            parity ^= 1;
        }
    }
    ptx::bulk_wait<0>();
}

// The field as a 4-D tensor [16-column group][tile of the group][z][columns of the tile] (TC = 16: one tile per group).
// Natural layout (x contiguous, z slowest): a group is 16 consecutive elements of a plane, rows nx*ny apart.
// Tile-blocked layout (`blocked`, see kernels.cuh): the nz rows of a group are contiguous (128 bytes each), so a
// group is one dense block of nz*128 bytes — DRAM pages are read and written whole.
bool make_field_map(CUtensorMap *map, const double *x, size_t plane, int nz, int tc, int box_rows, bool blocked) {
    const uint64_t dims[4] = {(uint64_t)tc, (uint64_t)nz, (uint64_t)(16 / tc), (uint64_t)(plane / 16)};
    const uint64_t strides[3] = {blocked ? (uint64_t)128 : (uint64_t)plane * sizeof(double), (uint64_t)tc * sizeof(double),
                                 blocked ? (uint64_t)nz * 128 : (uint64_t)128};
    const uint32_t box[4] = {(uint32_t)tc, (uint32_t)box_rows, 1, 1};
    return make_f64_map(map, x, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_NONE);
}

constexpr size_t SMEM_PER_SM = 228 * 1024, SMEM_CTA_RESERVED = 1024, SMEM_CTA_MAX = 227 * 1024;

// A launch shape: M rows per segment, TC columns per tile, at most MAXT threads per CTA, CTAS co-resident CTAs per SM
// (their barrier phases interleave), TS: regular coefficient table in shared memory.
struct Shape {
    int M, TC, MAXT, CTAS;
    bool TS;
};

// Launch geometry shared by the plain and the sharded launch.
struct ThomasGeom {
    int S, nbox, box_rows, buf_rows, nbuf, threads;
    size_t smem;
};
bool thomas_geometry(const Shape &sh, int nz, ThomasGeom &g) {
    const int row_bytes = sh.TC * (int)sizeof(double);
    int S = (nz + sh.M - 1) / sh.M;
    while ((S * sh.TC) % 32) ++S;                            // whole warps
    const int S4 = (S + 3) / 4 * 4;                          // the tables hold whole groups of 4 segments,
    if (S4 * sh.M > nz + THOMAS_TABLE_PAD) return false;     // nz + THOMAS_TABLE_PAD rows in all
    const int nbox = (nz + 255) / 256;                       // TMA boxes are at most 256 rows tall
    int box_rows = (nz + nbox - 1) / nbox;
    const int rows_128 = row_bytes >= 128 ? 1 : 128 / row_bytes;
    box_rows = (box_rows + rows_128 - 1) / rows_128 * rows_128;   // TMA wants 128-byte aligned shared-memory boxes
    // Shapes with several CTAs per SM keep only the rows the TMA boxes fill (>= nz): their segments may reach past the
    // buffer (kernel: `live`), which buys a third ring slot or the coefficient table in shared memory.  One-CTA shapes
    // have the room for all S*M rows and skip the predicates (their 16 warps run phase 1 together: issue-bound there;
    // 1024 rows: 1.00 -> 0.92 ms per 512 x 512 columns).
    const int buf_rows = (sh.CTAS > 1 || S * sh.M < nbox * box_rows) ? nbox * box_rows : S * sh.M;
    const size_t tile_bytes = (size_t)buf_rows * row_bytes;
    const size_t fixed = (size_t)6 * S * sh.TC * sizeof(double) + 128 + (sh.TS ? (size_t)S4 * sh.M * 32 : 0);
    size_t budget = SMEM_PER_SM / sh.CTAS - SMEM_CTA_RESERVED;
    if (budget > SMEM_CTA_MAX) budget = SMEM_CTA_MAX;
    if (budget < fixed + 2 * tile_bytes) return false;
    int nbuf = (int)((budget - fixed) / tile_bytes);
    if (nbuf > 3) nbuf = 3;
    // one-CTA shapes: a third ring slot would take the shared-memory carve-out to its maximum and leave the L1 too small for
    // the coefficient table (up to 35 KB) — measured equal at 840 / 900 rows, 7 % slower at 960 / 1008 rows
    if (sh.CTAS == 1 && nbuf > 2) nbuf = 2;
    if (sh.TC * S > sh.MAXT) return false;
    g = {S, nbox, box_rows, buf_rows, nbuf, sh.TC * S, (size_t)nbuf * tile_bytes + fixed};
    return true;
}

// `cols` = number of (kx,ky) columns of the field at `in` (nx*ny, or the rows a rank owns times nx).
// peers == nullptr: plain solve into the field x (same layout as `in`); else the sharded store of StorePeers.
// tab: the tables of thomas_onchip_tables; part = 0 / 1: the partition (blocked / natural launch shape) this launch is.
template <int M, int TC, int MAXT, int CTAS, bool SH, bool TS>
cudaError_t launch_m(const double *in, double *x, const ThomasPeers *peers, const double *tab, int part, const double *lamx, const double *lamy,
                     const double *wz, int nx, size_t cols, int nz, double shift0, int singular, bool blocked, int sms, cudaStream_t stream) {
    ThomasGeom g;
    if (!thomas_geometry(Shape{M, TC, MAXT, CTAS, TS}, nz, g)) return cudaErrorInvalidConfiguration;
    auto kern = thomas_onchip_kernel<M, TC, MAXT, CTAS, SH, TS>;
    static DeviceOnce configured;                            // per device, thread-safe (devonce.hpp)
    static OccupancyCache occupancy;
    cudaError_t e = configured.run([&] { return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CTA_MAX); });
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = occupancy.get(kern, g.threads, g.smem, &per_sm);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorInvalidConfiguration;
    CUtensorMap tmap;
    if (!make_field_map(&tmap, in, cols, nz, TC, g.box_rows, blocked)) return cudaErrorUnknown;
    const int ntiles = (int)(cols / TC);
    int grid = sms * per_sm;
    if (grid > ntiles) grid = ntiles;
    const size_t tab_block = 4 * ((size_t)nz + THOMAS_TABLE_PAD);
    tab += (size_t)(2 * part) * tab_block;                   // this partition's tables: regular, null
    const double *tab_null = tab + tab_block;
    if constexpr (SH) {
        StorePeers dst{};
        dst.npeers = peers->npeers;
        dst.group0 = peers->group0;
        int longest = 0;
        for (int r = 0; r <= peers->npeers; ++r) dst.k0[r] = peers->k0[r];
        for (int r = 0; r < peers->npeers; ++r) longest = peers->k0[r + 1] - peers->k0[r] > longest ? peers->k0[r + 1] - peers->k0[r] : longest;
        const int nb = (longest + 255) / 256;
        dst.box_rows = (longest + nb - 1) / nb;
        if (dst.box_rows & 1) ++dst.box_rows;                // even: 8-column rows stay 128-byte aligned in shared memory
        if (dst.box_rows < 1) dst.box_rows = 2;
        for (int r = 0; r < peers->npeers; ++r) {
            const int nzl = peers->k0[r + 1] - peers->k0[r];
            if (nzl <= 0) continue;                          // an empty slab receives nothing
            if ((peers->k0[r] & 1) && TC < 16) return cudaErrorInvalidValue;
            if (!make_field_map(&dst.map[r], peers->slab[r], peers->total_cols, nzl, TC, dst.box_rows, true)) return cudaErrorUnknown;
        }
        return launch_pdl(kern, dim3(grid), dim3(g.threads), g.smem, stream, tmap, dst, tab, tab_null, lamx, lamy, wz, nx, nz, g.S, g.nbuf,
                          g.box_rows, g.nbox, g.buf_rows, shift0, singular, ntiles);
    } else {
        StoreOne dst;
        if (!make_field_map(&dst.map, x, cols, nz, TC, g.box_rows, blocked)) return cudaErrorUnknown;
        return launch_pdl(kern, dim3(grid), dim3(g.threads), g.smem, stream, tmap, dst, tab, tab_null, lamx, lamy, wz, nx, nz, g.S, g.nbuf,
                          g.box_rows, g.nbox, g.buf_rows, shift0, singular, ntiles);
    }
}

}  // namespace

bool thomas_onchip_supported(int nx, int ny, int nz) {
    return ((size_t)nx * ny) % 16 == 0 && nz >= 2 && nz <= 1056;
}

namespace {

// The launch shape for columns of nz rows.  blocked_any: the field is tile-blocked, or a natural-layout launch asks for
// the same partition (tpt_solve_host, whose results equal tpt_solve's bit for bit).  allow4: 4-column tiles permitted.
// Measured on the box (profiles/): the sweep is bound by the LSU data pipe and the dependent FP64 chains of the 16 warps
// the register file admits per SM, so the shapes differ in wavefronts per row and in how well the phases of
// co-resident CTAs interleave.
Shape choose_shape(int nz, bool blocked_any, bool allow4) {
    // Short columns on the blocked layout: the 17-row / 8-column shape also wins below 257 rows wherever its segments fill
    // the column (at most 10 % padding rows: 64, 128, 192 rows — 512 x 512 columns x 128 rows: 0.139 -> 0.107 ms);
    // otherwise the 8- / 16-row shapes below (160, 224, 256 rows: measured equal or better)
    if (blocked_any && nz <= 204) {
        const int S = ((nz + 16) / 17 + 3) / 4 * 4;
        if (S * 17 * 10 <= 11 * nz) return {17, 8, 256, 2, false};
    }
    if (nz <= 128) return {8, 16, 256, 2, false};
    if (nz <= 256) return {16, 16, 256, 2, false};
    // 257 .. 800 rows on the blocked layout: narrow tiles, odd segment length (the segments of a warp then fall into
    // different banks: conflict-free), several CTAs per SM, at most 32 segments.  Segment length: the shortest of 17 / 19 /
    // 21 / 23 / 25 rows that covers the column (768^3: 0.709 -> 0.667 ms against one 384-thread CTA of 32-row segments),
    // unless another one leaves at least 3 % fewer padded rows — the padding is pure waste (416 rows: 0.400 -> 0.362 ms
    // with 21-row segments, 288 rows: 0.262 -> 0.240 ms with 25).
    if (blocked_any && nz <= 800) {
        int defM = 17;
        while (defM * 32 < nz) defM += 2;
        auto rows_of = [&](int M) { return ((nz + M - 1) / M + 3) / 4 * 4 * M; };
        int bestM = defM, bestRows = rows_of(defM);
        for (int M = defM + 2; M <= 25; M += 2)
            if (rows_of(M) * 100 < bestRows * 97 || (bestM != defM && rows_of(M) <= bestRows)) { bestRows = rows_of(M); bestM = M; }
        ThomasGeom g;
        // 4-column tiles, four CTAs of 4 warps per SM (same segments, so the same arithmetic): smaller barrier domains and
        // twice as many independent tile rings — where the segment count is a multiple of 8 anyway (no extra padding)
        // and M <= 19 (measured, interleaved runs at 512 x 512 columns: 384 / 448 rows 7-8 % faster, 512 rows 4 %, 608 rows
        // 3.5 %, 576 rows equal; 21-row segments — 640, 672 rows — equal or slower).
        // The coefficient table goes to shared memory where it fits beside two tile buffers and the CTAs fill the register
        // file anyway (512 threads per SM; below that a smaller footprint lets more CTAs in: 320 rows 0.29 vs 0.35 ms):
        // 512 rows with 4-column tiles 0.440 vs 0.454 ms, with 8-column tiles 0.458 vs 0.476 ms.
        const int segs = (nz + bestM - 1) / bestM;
        const int S8 = (segs + 3) / 4 * 4;
        const bool ts_ok = S8 * 16 >= 512;
        if (allow4 && bestM <= 19 && S8 == (segs + 7) / 8 * 8) {
            Shape s4{bestM, 4, 128, 4, ts_ok};
            if (thomas_geometry(s4, nz, g)) return s4;
            s4.TS = false;
            if (thomas_geometry(s4, nz, g)) return s4;
        }
        Shape s8{bestM, 8, 256, 2, ts_ok};
        if (thomas_geometry(s8, nz, g)) return s8;
        s8.TS = false;
        return s8;
    }
    if (nz <= 512) return {16, 16, 512, 1, false};
    if (nz <= 768) return {32, 16, 384, 1, false};
    // up to 1056 rows: 8-column tiles of 17-row segments, 512 threads (16 warps), two 68 KB buffers, one CTA per SM
    // (33-row segments with 256 threads and 242 registers: 4.25 instead of 3.69 ms at 1024^3)
    // 801 .. 1008 rows: 21-row segments (at most 48 per column, 384 threads) — measured 0.84 / 0.86 / 1.05 / 1.05 ms at
    // 840 / 900 / 960 / 992 rows against 0.94 / 1.07 / 1.10 / 1.11 ms with 17-row segments (512 x 512 columns); from 1009
    // rows on the 17-row, 64-segment shape wins (1024 rows: 0.97 vs 1.18 ms)
    if (nz <= 1008) return {21, 8, 416, 1, false};
    return {17, 8, 512, 1, false};
}

template <bool SH>
cudaError_t dispatch(const double *in, double *x, const ThomasPeers *peers, const double *tab, const double *lamx, const double *lamy,
                     const double *wz, int nx, size_t cols, int nz, double shift0, int singular, bool blocked, bool blocked_shape,
                     int sms, cudaStream_t stream) {
    const bool blocked_any = blocked || blocked_shape;
    // the sharded store cuts tiles at the z-slab boundaries (even numbers): 4-column rows would lose their 128-byte alignment
    const Shape sh = choose_shape(nz, blocked_any, !SH);
    const int part = blocked_any ? 0 : 1;
#define TPT_TRY(M_, TC_, MAXT_, CTAS_, TS_)                                                                                    \
    if (sh.M == M_ && sh.TC == TC_ && sh.MAXT == MAXT_ && sh.CTAS == CTAS_ && sh.TS == TS_)                                    \
        return launch_m<M_, TC_, MAXT_, CTAS_, SH, TS_>(in, x, peers, tab, part, lamx, lamy, wz, nx, cols, nz, shift0, singular, \
                                                        blocked, sms, stream);
    TPT_TRY(17, 8, 256, 2, false) TPT_TRY(19, 8, 256, 2, false) TPT_TRY(21, 8, 256, 2, false) TPT_TRY(23, 8, 256, 2, false)
    TPT_TRY(25, 8, 256, 2, false)
    TPT_TRY(17, 8, 256, 2, true) TPT_TRY(19, 8, 256, 2, true) TPT_TRY(21, 8, 256, 2, true)   // 23, 25: never fits
    if constexpr (!SH) {
        TPT_TRY(17, 4, 128, 4, true) TPT_TRY(17, 4, 128, 4, false) TPT_TRY(19, 4, 128, 4, false)   // 19 rows: the table never fits
    }
    TPT_TRY(8, 16, 256, 2, false) TPT_TRY(16, 16, 256, 2, false) TPT_TRY(16, 16, 512, 1, false) TPT_TRY(32, 16, 384, 1, false)
    TPT_TRY(21, 8, 416, 1, false) TPT_TRY(17, 8, 512, 1, false)
#undef TPT_TRY
    return cudaErrorInvalidConfiguration;
}
}  // namespace

cudaError_t launch_thomas_onchip(const double *in, double *x, const double *tab, const double *lamx, const double *lamy, const double *wz,
                                 int nx, int ny, int nz, double shift0, int singular, bool blocked, bool blocked_shape, int sms,
                                 cudaStream_t stream) {
    if (!thomas_onchip_supported(nx, ny, nz)) return cudaErrorInvalidValue;
    return dispatch<false>(in, x, nullptr, tab, lamx, lamy, wz, nx, (size_t)nx * ny, nz, shift0, singular, blocked, blocked_shape, sms, stream);
}

cudaError_t launch_thomas_onchip_sharded(const double *in, const ThomasPeers &peers, const double *tab, const double *lamx,
                                         const double *lamy_owned, const double *wz, int nx, int rows, int nz, double shift0,
                                         int singular, int sms, cudaStream_t stream) {
    if (rows < 1 || nx % 16 || nz < 2 || nz > 1056 || peers.npeers < 1 || peers.npeers > MAX_PEERS) return cudaErrorInvalidValue;
    return dispatch<true>(in, nullptr, &peers, tab, lamx, lamy_owned, wz, nx, (size_t)nx * rows, nz, shift0, singular, true, false, sms, stream);
}

// The launch geometry dispatch() would use, for inspection (tests sweep every nz): out = { M, columns per tile, thread limit,
// CTAs per SM, table in shared memory, S, TMA boxes per tile, rows per box, rows per tile buffer, ring slots, threads, dynamic
// shared memory bytes }.  false: this nz has no on-chip shape in that layout.
bool thomas_onchip_geometry(int nz, bool blocked_any, bool sharded, int out[12]) {
    if (nz < 2 || nz > 1056) return false;
    const Shape sh = choose_shape(nz, blocked_any, !sharded);
    ThomasGeom g;
    if (!thomas_geometry(sh, nz, g)) return false;
    const int v[12] = {sh.M, sh.TC, sh.MAXT, sh.CTAS, sh.TS ? 1 : 0, g.S, g.nbox, g.box_rows, g.buf_rows, g.nbuf, g.threads, (int)g.smem};
    for (int i = 0; i < 12; ++i) out[i] = v[i];
    return true;
}

// Host side of the coefficient tables: rows [a_k c_{k-1}, b_k, a_k, c_k], padded with decoupled rows
// [0, -1, 0, 0] (pivot -1 + s < 0 for every mode since s <= 0); the second table is the null column's, with the
// last equation replaced by "-x = p" (the kernel zeroes p there): PAPER.md:219.  Both are stored once per partition the
// launches of this nz can have (0: blocked layout / blocked_shape, 1: natural layout), in the order the kernel reads
// them: row t of segment seg — row seg M + t of the column — at (((seg / 4) M + t) 4 + seg % 4) * 4 (groups of 4 segments,
// row-interleaved).  Four blocks of 4 (nz + THOMAS_TABLE_PAD) doubles.
void thomas_onchip_tables(int nz, const double *a, const double *b, const double *c, std::vector<double> &out, const double *b_null) {
    const size_t rows = (size_t)nz + THOMAS_TABLE_PAD;
    std::vector<double> nat(8 * rows, 0.0);
    for (int v = 0; v < 2; ++v) {
        double *t = nat.data() + (size_t)v * 4 * rows;
        for (size_t k = 0; k < rows; ++k) t[4 * k + 1] = -1.0;
        for (int k = 0; k < nz; ++k) {
            t[4 * k] = k > 0 ? a[k] * c[k - 1] : 0.0;
            t[4 * k + 1] = (v == 1 && b_null) ? b_null[k] : b[k];
            t[4 * k + 2] = a[k];
            t[4 * k + 3] = c[k];
        }
        if (v == 1) {
            double *last = t + 4 * (size_t)(nz - 1);
            last[0] = 0.0; last[1] = -1.0; last[2] = 0.0; last[3] = 0.0;
        }
    }
    out.assign(16 * rows, 0.0);
    for (int part = 0; part < 2; ++part) {
        const Shape sh = choose_shape(nz, part == 0, true);    // 4- and 8-column shapes of one nz share M and S
        ThomasGeom g;
        if (!thomas_geometry(sh, nz, g)) continue;
        for (int v = 0; v < 2; ++v) {
            const double *src = nat.data() + (size_t)v * 4 * rows;
            double *dst = out.data() + (size_t)(2 * part + v) * 4 * rows;
            for (int seg = 0; seg < g.S; ++seg)
                for (int t = 0; t < sh.M; ++t)
                    for (int j = 0; j < 4; ++j)
                        dst[(((size_t)(seg >> 2) * sh.M + t) * 4 + (seg & 3)) * 4 + j] = src[((size_t)seg * sh.M + t) * 4 + j];
        }
    }
}

}  // namespace tpt
