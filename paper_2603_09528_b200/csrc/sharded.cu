// sharded.cu — the solve sharded across the GPUs of one NVLink domain (PAPER.md:197-207 pencil layouts
// and collective transposes, Algorithm 1 steps 2, 4, 6, 8 at PAPER.md:235-245).
//
// The paper transposes between x-, y- and z-aligned pencils with four all-to-alls per solve.  Here a rank owns
//   * a z-SLAB of the physical field, planes [k0_r, k0_{r+1}): steps 2.1, 2.2, 2.4, 2.5 act plane by plane (Eq. 10, 12), so
//     both x and y transforms are local to it — two of the paper's four transposes disappear;
//   * a block of y-MODE rows [m0_q, m0_{q+1}) x all kx x all z of the mode-space field for step 2.3 (Eq. 11).
// The two remaining exchanges are not collectives but the stores of kernels that touch the data anyway:
//   exchange 1  the forward-y GEMM epilogue writes every mode row straight into its owner's memory (GemmArgs::peerC),
//   exchange 2  the sweep's TMA store writes rows [k0_r, k0_{r+1}) of every solved tile into rank r's slab buffer
//               (StorePeers in thomas_onchip.cu),
// both through peer-mapped pointers (NVLink 5 / NVSwitch; writes are posted, so the links run while the tensor pipe /
// HBM work continues).  Each element crosses NVLink once per exchange: 8 * pts * (P-1) / P^2 bytes per rank and direction.
//
// Memory per rank ("symmetric" allocation, same offsets on every rank, one IPC handle):
//   [ mode buffer: rows_max * nx * nz doubles, tile-blocked ((m_loc * nx/16 + i/16) * nz + k) * 16 + i%16 ]
//   [ slab buffer: ny * nx * nzl_max doubles, tile-blocked ((m * nx/16 + i/16) * nzl_r + k_loc) * 16 + i%16 ]
//   [ signal pad:  one 64-bit epoch flag per peer ]
// Ordering across ranks: two barriers per solve (after exchange 1, after exchange 2).  tpt_solve_sharded uses a
// device-side flag barrier over the signal pads; tpt_shard_solve_phase enqueues one phase without any waiting kernel,
// for callers that order the phases themselves (virtual ranks on one device: the tests and the one-GPU bench leg).
#include <cuda_runtime.h>

#include <cstdint>
#include <cstring>
#include <new>

#include "kernels.cuh"
#include "plan.hpp"

struct tpt_shard {
    tpt_plan *plan = nullptr;          // full-grid plan: matrices, tables; its workspace holds one z-slab
    tpt_shard_layout_t lay{};
    int k0[tpt::MAX_PEERS + 1] = {};   // z-slab boundaries of every rank
    int m0[tpt::MAX_PEERS + 1] = {};   // mode-row boundaries of every rank
    size_t mode_off = 0, slab_off = 0, pad_off = 0;
    unsigned char *sym = nullptr;                      // own symmetric allocation
    unsigned char *peer[tpt::MAX_PEERS] = {};          // every rank's allocation as mapped into this process
    bool opened[tpt::MAX_PEERS] = {};                  // mapping came from cudaIpcOpenMemHandle
    bool peers_set = false;
    unsigned long long epoch = 0;                      // barriers passed so far
    int launches_last = 0;
};

namespace {

constexpr size_t PAD_BYTES = 4096;
size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// plane split in units of two planes (even boundaries: thomas_onchip.cu StorePeers), row split in units of 16 rows
// (a GEMM k-slab / a 16-row epilogue group never straddles two owners)
int plane_start(int nz, int r, int P) {
    const long long hz = (nz + 1) / 2;
    const long long k = 2 * (hz * r / P);
    return (int)(k > nz ? nz : k);
}
int row_start(int ny, int q, int P) { return 16 * (int)((long long)(ny / 16) * q / P); }

// the GEMM shapes (nx, ny multiples of 128) cover every transform choice; tpt_shard_create_ex accepts a fast y transform
// on any supported power of two (ny / 16 >= P)
bool layout_ok(int P, int nx, int ny, int nz) {
    return P >= 1 && P <= tpt::MAX_PEERS && nx >= 128 && nx % 128 == 0 && ny >= 16 && ny % 16 == 0 && nz >= 2 * P &&
           ny / 16 >= P && nz <= 1056;
}

struct PadPtrs { unsigned long long *pad[tpt::MAX_PEERS]; };

// Flag barrier over the signal pads: thread t of rank `rank` tells rank t "rank `rank` has reached epoch e" and waits
// until rank t has said the same here.  Epochs only grow, so a rank that races ahead to its next barrier cannot be missed.
// The fence orders every earlier write of this rank (the exchange stores of the kernel before it on the stream — complete,
// since kernels on one stream run in order) before the flag.
__device__ void flag_barrier(const PadPtrs &pads, int rank, int npeers, unsigned long long epoch) {
    const int t = threadIdx.x;
    if (t >= npeers) return;
    __threadfence_system();
    asm volatile("st.release.sys.global.u64 [%0], %1;\n" ::"l"(pads.pad[t] + rank), "l"(epoch) : "memory");
    unsigned long long seen;
    do {
        asm volatile("ld.acquire.sys.global.u64 %0, [%1];\n" : "=l"(seen) : "l"(pads.pad[rank] + t) : "memory");
    } while (seen < epoch);
    __threadfence_system();
}

__global__ void shard_barrier_kernel(PadPtrs pads, int rank, int npeers, unsigned long long epoch) {
    flag_barrier(pads, rank, npeers, epoch);
}

// All ranks of a set of virtual ranks (one device) in ONE cooperative launch, block r acting as rank r: kernels that wait
// on one another must not be separate launches on one GPU (nothing guarantees they run at the same time), co-resident
// blocks of one cooperative grid may.  Same flag code as above.
struct EpochList { unsigned long long e[tpt::MAX_PEERS]; };
__global__ void shard_barrier_all_kernel(PadPtrs pads, int npeers, EpochList epochs) {
    flag_barrier(pads, blockIdx.x, npeers, epochs.e[blockIdx.x]);
}

void free_shard(tpt_shard *s) {
    if (!s) return;
    for (int r = 0; r < tpt::MAX_PEERS; ++r)
        if (s->opened[r] && s->peer[r]) cudaIpcCloseMemHandle(s->peer[r]);
    cudaFree(s->sym);
    if (s->plan) tpt_plan_destroy(s->plan);
    delete s;
}

double *mode_of(const tpt_shard *s, int r) { return reinterpret_cast<double *>(s->peer[r] + s->mode_off); }
double *slab_of(const tpt_shard *s, int r) { return reinterpret_cast<double *>(s->peer[r] + s->slab_off); }

int barrier(tpt_shard *s, cudaStream_t st) {
    PadPtrs pp{};
    for (int r = 0; r < s->lay.nranks; ++r) pp.pad[r] = reinterpret_cast<unsigned long long *>(s->peer[r] + s->pad_off);
    ++s->epoch;
    shard_barrier_kernel<<<1, 32, 0, st>>>(pp, s->lay.rank, s->lay.nranks, s->epoch);
    return cudaGetLastError() == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

// phase 0: steps 2.1, 2.2 on the own z-slab; mode rows pushed to their owners (exchange 1)
int phase_forward(tpt_shard *s, const double *rhs, cudaStream_t st, int *launches) {
    tpt_plan *p = s->plan;
    const int r = s->lay.rank, P = s->lay.nranks, nzl = s->lay.k1 - s->lay.k0;
    double *W = p->d_work;
    const double *cur = rhs;
    if (p->dirs & 1) {
        int rc = tpt::detail::run_slot(p, TPT_K_FWD_X, rhs, W, st, launches, 0, nzl);
        if (rc != TPT_OK) return rc;
        cur = W;
    }
    if (p->transform[1] == TPT_TRANSFORM_FFT) {
        // fast y transform: the same scatter from the kernel's own stores (row `slot` of the blocked mode buffer of its owner)
        tpt::FftArgs a{};
        a.in = cur; a.out = nullptr;
        a.tables = p->d_fft[1];
        a.dir = 1; a.inverse = 0; a.bc = p->bc[1];
        a.nx = p->nx; a.ny = p->ny; a.planes = nzl;
        a.s0 = p->fft_s[1][0]; a.s1 = p->fft_s[1][1];
        a.blocked = 1; a.nz = p->nz; a.k0 = s->k0[r];
        a.npeers = P;
        const int64_t row_stride = (int64_t)p->nx * p->nz;          // elements between mode rows of a blocked buffer
        for (int q = 0; q < P; ++q)
            a.peer_out[q] = reinterpret_cast<double *>(reinterpret_cast<intptr_t>(mode_of(s, q)) -
                                                       (intptr_t)s->m0[q] * row_stride * (intptr_t)sizeof(double));
        ++*launches;
        return tpt::launch_fft(a, st) == cudaSuccess ? TPT_OK : TPT_ECUDA;
    }
    tpt::GemmArgs g{};
    g.A = p->d_yfwd; g.lda = p->ny; g.strideA = 0;
    g.M = p->ny; g.N = p->nx; g.K = p->ny;
    g.B = cur; g.ldb = p->nx; g.strideB = (int64_t)p->nx * p->ny;
    g.batch = nzl;
    g.C = nullptr; g.ldc = (int64_t)p->nx * p->nz; g.strideC = 16; g.ldgC = (int64_t)16 * p->nz;
    g.npeers = P;
    for (int q = 0; q < P; ++q) {
        // element (row m, column i, local plane b) -> owner q's mode buffer at ((m - m0_q) nx/16 + i/16) nz + k0_r + b) 16 + i%16
        const intptr_t shift = ((intptr_t)16 * s->k0[r] - (intptr_t)s->m0[q] * g.ldc) * (intptr_t)sizeof(double);
        g.peerC[q] = reinterpret_cast<double *>(reinterpret_cast<intptr_t>(mode_of(s, q)) + shift);
    }
    if (!tpt::gemm_tma_supported(g)) return TPT_EINVAL;
    ++*launches;
    return tpt::launch_gemm_tma(g, p->sms, st) == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

// phase 1: step 2.3 on the owned mode rows; solution rows pushed to the z-slab owners (exchange 2)
int phase_sweep(tpt_shard *s, cudaStream_t st, int *launches) {
    tpt_plan *p = s->plan;
    const int r = s->lay.rank, P = s->lay.nranks;
    tpt::ThomasPeers tp;
    tp.npeers = P;
    for (int q = 0; q <= P; ++q) tp.k0[q] = s->k0[q];
    for (int q = 0; q < P; ++q) tp.slab[q] = slab_of(s, q);
    tp.total_cols = (size_t)p->nx * p->ny;
    tp.group0 = (int)((int64_t)s->m0[r] * p->nx / 16);
    ++*launches;
    cudaError_t e = tpt::launch_thomas_onchip_sharded(mode_of(s, r), tp, p->d_abc, p->d_lamx, p->d_lamy + s->m0[r], p->d_wz, p->nx,
                                                      s->m0[r + 1] - s->m0[r], p->nz, p->shift0, p->singular && s->m0[r] == 0,
                                                      p->sms, st);
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

// phase 2: steps 2.4, 2.5 on the own z-slab (its mode-space values were delivered into the slab buffer)
int phase_inverse(tpt_shard *s, double *out, cudaStream_t st, int *launches) {
    tpt_plan *p = s->plan;
    const int r = s->lay.rank, nzl = s->lay.k1 - s->lay.k0;
    double *W = p->d_work;
    double *dst = (p->dirs & 1) ? W : out;
    if (p->transform[1] == TPT_TRANSFORM_FFT) {
        tpt::FftArgs a{};
        a.in = slab_of(s, r); a.out = dst;
        a.tables = p->d_fft[1];
        a.dir = 1; a.inverse = 1; a.bc = p->bc[1];
        a.nx = p->nx; a.ny = p->ny; a.planes = nzl;
        a.s0 = p->fft_s[1][2]; a.s1 = p->fft_s[1][3];
        a.blocked = 1; a.nz = nzl; a.k0 = 0;                          // the slab buffer is blocked over the rank's own planes
        ++*launches;
        if (tpt::launch_fft(a, st) != cudaSuccess) return TPT_ECUDA;
        if (p->dirs & 1) return tpt::detail::run_slot(p, TPT_K_INV_X, W, out, st, launches, 0, nzl);
        return TPT_OK;
    }
    tpt::GemmArgs g{};
    g.A = p->d_yinv; g.lda = p->ny; g.strideA = 0;
    g.M = p->ny; g.N = p->nx; g.K = p->ny;
    g.B = slab_of(s, r); g.ldb = (int64_t)p->nx * nzl; g.strideB = 16; g.ldgB = (int64_t)16 * nzl;
    g.batch = nzl;
    g.C = dst; g.ldc = p->nx; g.strideC = (int64_t)p->nx * p->ny;
    if (!tpt::gemm_tma_supported(g)) return TPT_EINVAL;
    ++*launches;
    if (tpt::launch_gemm_tma(g, p->sms, st) != cudaSuccess) return TPT_ECUDA;
    if (p->dirs & 1) return tpt::detail::run_slot(p, TPT_K_INV_X, W, out, st, launches, 0, nzl);
    return TPT_OK;
}

bool aligned16(const void *q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; }

}  // namespace

extern "C" {

int tpt_shard_layout(int nranks, int rank, int nx, int ny, int nz, tpt_shard_layout_t *out) {
    if (!out || rank < 0 || rank >= nranks || !layout_ok(nranks, nx, ny, nz)) return TPT_EINVAL;
    tpt_shard_layout_t l{};
    l.rank = rank; l.nranks = nranks;
    l.k0 = plane_start(nz, rank, nranks); l.k1 = plane_start(nz, rank + 1, nranks);
    l.m0 = row_start(ny, rank, nranks); l.m1 = row_start(ny, rank + 1, nranks);
    int rows_max = 0, nzl_max = 0;
    for (int q = 0; q < nranks; ++q) {
        const int rows = row_start(ny, q + 1, nranks) - row_start(ny, q, nranks);
        const int nzl = plane_start(nz, q + 1, nranks) - plane_start(nz, q, nranks);
        rows_max = rows > rows_max ? rows : rows_max;
        nzl_max = nzl > nzl_max ? nzl : nzl_max;
    }
    l.mode_bytes = (size_t)rows_max * nx * nz * sizeof(double);
    l.slab_bytes = (size_t)ny * nx * nzl_max * sizeof(double);
    l.sym_bytes = align_up(l.mode_bytes, 256) + align_up(l.slab_bytes, 256) + PAD_BYTES;
    l.slab_points = (size_t)nx * ny * (l.k1 - l.k0);
    l.nvlink_bytes_per_solve = 2 * sizeof(double) * ((size_t)nx * (l.m1 - l.m0) * (size_t)(nz - (l.k1 - l.k0)));
    *out = l;
    return TPT_OK;
}

int tpt_shard_create(tpt_shard **shard_out, int rank, int nranks, int nx, int ny, int nz, const double *xf, const double *yf,
                     const double *zf, const int bc[3], double helmholtz_alpha, int transform_x) {
    const int transform[2] = {transform_x, TPT_TRANSFORM_GEMM};
    return tpt_shard_create_ex(shard_out, rank, nranks, nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha, transform);
}

int tpt_shard_create_ex(tpt_shard **shard_out, int rank, int nranks, int nx, int ny, int nz, const double *xf, const double *yf,
                        const double *zf, const int bc[3], double helmholtz_alpha, const int transform_xy[2]) {
    if (!shard_out || !bc || !transform_xy || bc[2] == TPT_BC_PERIODIC) return TPT_EINVAL;   // (the cyclic correction is not sharded)
    if (transform_xy[1] != TPT_TRANSFORM_FFT && ny % 128) return TPT_EINVAL;                 // the GEMM's exchange needs full 128-row tiles
    tpt_shard_layout_t lay;
    int rc = tpt_shard_layout(nranks, rank, nx, ny, nz, &lay);
    if (rc != TPT_OK) return rc;
    tpt_shard *s = new (std::nothrow) tpt_shard();
    if (!s) return TPT_ENOMEM;
    s->lay = lay;
    for (int q = 0; q <= nranks; ++q) { s->k0[q] = plane_start(nz, q, nranks); s->m0[q] = row_start(ny, q, nranks); }
    s->mode_off = 0;
    s->slab_off = align_up(lay.mode_bytes, 256);
    s->pad_off = s->slab_off + align_up(lay.slab_bytes, 256);
    const int transform[2] = {transform_xy[0], transform_xy[1]};  // the y transform (TMA GEMM or fast transform) carries exchange 1
    rc = tpt::detail::plan_create_sized(&s->plan, nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha, TPT_DIRS_XYZ, transform,
                                        lay.slab_bytes / sizeof(double));
    if (rc != TPT_OK) { free_shard(s); return rc; }
    cudaError_t e = cudaMalloc(&s->sym, lay.sym_bytes);
    if (e == cudaSuccess) e = cudaMemset(s->sym + s->pad_off, 0, PAD_BYTES);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        cudaGetLastError();
        free_shard(s);
        return e == cudaErrorMemoryAllocation ? TPT_ENOMEM : TPT_ECUDA;
    }
    s->peer[rank] = s->sym;
    if (nranks == 1) s->peers_set = true;
    *shard_out = s;
    return TPT_OK;
}

int tpt_shard_get_layout(const tpt_shard *s, tpt_shard_layout_t *out) {
    if (!s || !out) return TPT_EINVAL;
    *out = s->lay;
    return TPT_OK;
}

int tpt_shard_sym(const tpt_shard *s, void **sym_dev_out, size_t *bytes_out) {
    if (!s || !sym_dev_out) return TPT_EINVAL;
    *sym_dev_out = s->sym;
    if (bytes_out) *bytes_out = s->lay.sym_bytes;
    return TPT_OK;
}

int tpt_shard_set_peers(tpt_shard *s, void *const *sym_dev) {
    if (!s || !sym_dev) return TPT_EINVAL;
    for (int r = 0; r < s->lay.nranks; ++r) {
        if (!sym_dev[r] || !aligned16(sym_dev[r])) return TPT_EINVAL;
        if (r == s->lay.rank && sym_dev[r] != s->sym) return TPT_EINVAL;
    }
    for (int r = 0; r < s->lay.nranks; ++r) {
        if (s->opened[r]) { cudaIpcCloseMemHandle(s->peer[r]); s->opened[r] = false; }
        s->peer[r] = static_cast<unsigned char *>(sym_dev[r]);
    }
    s->peers_set = true;
    return TPT_OK;
}

int tpt_shard_ipc_export(const tpt_shard *s, void *handle_out) {
    if (!s || !handle_out) return TPT_EINVAL;
    static_assert(sizeof(cudaIpcMemHandle_t) == TPT_IPC_HANDLE_BYTES, "IPC handle size");
    cudaIpcMemHandle_t h;
    if (cudaIpcGetMemHandle(&h, s->sym) != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
    std::memcpy(handle_out, &h, sizeof(h));
    return TPT_OK;
}

int tpt_shard_ipc_import(tpt_shard *s, const void *handles) {
    if (!s || !handles || !tpt::detail::on_plan_device(s->plan)) return TPT_EINVAL;
    for (int r = 0; r < s->lay.nranks; ++r) {
        if (r == s->lay.rank) continue;
        if (s->opened[r]) { cudaIpcCloseMemHandle(s->peer[r]); s->opened[r] = false; s->peer[r] = nullptr; }
        cudaIpcMemHandle_t h;
        std::memcpy(&h, static_cast<const unsigned char *>(handles) + (size_t)r * sizeof(h), sizeof(h));
        void *ptr = nullptr;
        if (cudaIpcOpenMemHandle(&ptr, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
        s->peer[r] = static_cast<unsigned char *>(ptr);
        s->opened[r] = true;
    }
    s->peer[s->lay.rank] = s->sym;
    s->peers_set = true;
    return TPT_OK;
}

int tpt_shard_solve_phase(tpt_shard *s, int phase, const double *rhs_slab_dev, double *out_slab_dev, void *cuda_stream) {
    if (!s || phase < 0 || phase > 2 || !s->peers_set || !tpt::detail::on_plan_device(s->plan)) return TPT_EINVAL;
    if (phase == 0 && (!rhs_slab_dev || !aligned16(rhs_slab_dev))) return TPT_EINVAL;
    if (phase == 2 && (!out_slab_dev || !aligned16(out_slab_dev))) return TPT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0;
    int rc = phase == 0 ? phase_forward(s, rhs_slab_dev, st, &launches)
           : phase == 1 ? phase_sweep(s, st, &launches) : phase_inverse(s, out_slab_dev, st, &launches);
    s->launches_last = launches;
    return rc;
}

int tpt_shard_barrier(tpt_shard *s, void *cuda_stream) {
    if (!s || !s->peers_set || !tpt::detail::on_plan_device(s->plan)) return TPT_EINVAL;
    return barrier(s, static_cast<cudaStream_t>(cuda_stream));
}

int tpt_shard_barrier_all(tpt_shard *const *shards, int n, void *cuda_stream) {
    if (!shards || n < 1 || n > tpt::MAX_PEERS) return TPT_EINVAL;
    PadPtrs pp{};
    EpochList ep{};
    for (int r = 0; r < n; ++r) {
        tpt_shard *s = shards[r];
        if (!s || !s->peers_set || s->lay.nranks != n || s->lay.rank != r || !tpt::detail::on_plan_device(s->plan)) return TPT_EINVAL;
        pp.pad[r] = reinterpret_cast<unsigned long long *>(s->sym + s->pad_off);
        if (s->peer[r] != s->sym) return TPT_EINVAL;
    }
    for (int r = 0; r < n; ++r)
        for (int q = 0; q < n; ++q)
            if (shards[r]->peer[q] != shards[q]->sym) return TPT_EINVAL;     // virtual ranks: every peer is a local shard
    for (int r = 0; r < n; ++r) ep.e[r] = ++shards[r]->epoch;
    int np = n;
    void *args[] = {&pp, &np, &ep};
    cudaError_t e = cudaLaunchCooperativeKernel(reinterpret_cast<void *>(shard_barrier_all_kernel), dim3(n), dim3(32), args, 0,
                                                static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) { cudaGetLastError(); return TPT_ECUDA; }
    return TPT_OK;
}

int tpt_solve_sharded(tpt_shard *s, const double *rhs_slab_dev, double *out_slab_dev, void *cuda_stream) {
    if (!s || !rhs_slab_dev || !out_slab_dev || !aligned16(rhs_slab_dev) || !aligned16(out_slab_dev) || !s->peers_set ||
        !tpt::detail::on_plan_device(s->plan))
        return TPT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0;
    int rc = phase_forward(s, rhs_slab_dev, st, &launches);
    if (rc == TPT_OK) rc = barrier(s, st);          // every rank's mode rows have arrived
    if (rc == TPT_OK) rc = phase_sweep(s, st, &launches);
    if (rc == TPT_OK) rc = barrier(s, st);          // every rank's slab rows have arrived (and every mode buffer is free again)
    if (rc == TPT_OK) rc = phase_inverse(s, out_slab_dev, st, &launches);
    s->launches_last = launches + 2;
    return rc;
}

int tpt_shard_launches(const tpt_shard *s) { return s ? s->launches_last : TPT_EINVAL; }

int tpt_shard_destroy(tpt_shard *s) {
    if (!s) return TPT_OK;
    cudaError_t e = cudaDeviceSynchronize();
    free_shard(s);
    return e == cudaSuccess ? TPT_OK : TPT_ECUDA;
}

}  // extern "C"
