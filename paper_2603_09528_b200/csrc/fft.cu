// fft.cu — the eigenbasis transforms of a UNIFORM direction by fast transforms instead of GEMMs ("a
// uniform direction may use either FFT-based transforms or numerical eigenbasis transforms evaluated with GEMM",
// :211 "for a uniform direction, the analytical eigenvalues are stored", :221 O(N log N) per line).
//
// On a uniform direction the eigenvectors of the 1-D operator (Eq. 3-5 with the boundary rows of DESIGN.md A3) are
// known in closed form:   Neumann    q_k(i) ~ cos(pi k (2i+1) / 2N)            (DCT-II / DCT-III pair)
//                         Dirichlet  q_k(i) ~ sin(pi (k+1) (2i+1) / 2N)        (DST-II / DST-III pair)
//                         periodic   1, cos(2 pi j i / N), sin(2 pi j i / N), (-1)^i   (real DFT)
// so  p^ = Q~^T D^{1/2} f  and  phi = D^{-1/2} Q~ x^  (Eq. 10, 12) are one complex FFT of length N per PAIR of lines:
//   * two real lines ride in the real and imaginary parts of one complex sequence and are untangled afterwards
//     (V1_k = (Z_k + conj Z_{N-k})/2, V2_k = (Z_k - conj Z_{N-k})/2i);
//   * the cosine transforms use Makhoul's reordering v_n = f_{2n}, v_{N-1-n} = f_{2n+1}, C_k = Re(e^{-i pi k/2N} V_k);
//     the sine transforms are cosine transforms of (-1)^i f_i read backwards; the inverse transforms run the same
//     steps in reverse (Hermitian-symmetrised coefficients -> inverse FFT -> real part);
//   * the FFT is a Stockham autosort FFT in shared memory (radix 8/4/2 passes, ping-pong buffers, one barrier per
//     pass); a CTA owns several pairs of lines: contiguous rows for the x direction, a 16-column tile (128-byte rows)
//     for the y direction, so both directions run in the field's native layout without transposes.
// HBM-bound: 16 B/pt (read once, write once) against 2N flop/pt for the GEMM form.  N = 2^m, 16 <= N <= 2048.
#include "devonce.hpp"
#include "kernels.cuh"

namespace tpt {

namespace {

struct cplx { double x, y; };
__device__ __forceinline__ cplx operator+(cplx a, cplx b) { return {a.x + b.x, a.y + b.y}; }
__device__ __forceinline__ cplx operator-(cplx a, cplx b) { return {a.x - b.x, a.y - b.y}; }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return {fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x)}; }
// multiply by -i (forward) or +i (inverse)
template <int INV>
__device__ __forceinline__ cplx mul_mi(cplx a) { return INV ? cplx{-a.y, a.x} : cplx{a.y, -a.x}; }

template <int INV>
__device__ __forceinline__ void fft2(cplx *v) {
    const cplx a = v[0], b = v[1];
    v[0] = a + b;
    v[1] = a - b;
}
template <int INV>
__device__ __forceinline__ void fft4(cplx &v0, cplx &v1, cplx &v2, cplx &v3) {
    const cplx t0 = v0 + v2, t1 = v0 - v2, t2 = v1 + v3, t3 = mul_mi<INV>(v1 - v3);
    v0 = t0 + t2;
    v1 = t1 + t3;
    v2 = t0 - t2;
    v3 = t1 - t3;
}
template <int INV>
__device__ __forceinline__ void fft8(cplx *v) {
    fft4<INV>(v[0], v[2], v[4], v[6]);      // even inputs -> E_0..E_3 in v[0], v[2], v[4], v[6]
    fft4<INV>(v[1], v[3], v[5], v[7]);      // odd inputs  -> O_0..O_3 in v[1], v[3], v[5], v[7]
    constexpr double h = 0.70710678118654752440;
    const cplx o0 = v[1];
    const cplx o1 = INV ? cplx{h * (v[3].x - v[3].y), h * (v[3].x + v[3].y)} : cplx{h * (v[3].x + v[3].y), h * (v[3].y - v[3].x)};
    const cplx o2 = mul_mi<INV>(v[5]);
    const cplx o3 = INV ? cplx{-h * (v[7].x + v[7].y), h * (v[7].x - v[7].y)} : cplx{h * (v[7].y - v[7].x), -h * (v[7].x + v[7].y)};
    const cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    v[0] = e0 + o0; v[4] = e0 - o0;
    v[1] = e1 + o1; v[5] = e1 - o1;
    v[2] = e2 + o2; v[6] = e2 - o2;
    v[3] = e3 + o3; v[7] = e3 - o3;
}

// shared-memory index with one padding element per 8 (keeps the stride-R stores of the first pass conflict-free)
__device__ __forceinline__ int pad(int i) { return i + (i >> 3); }

// One Stockham pass of radix R over `pairs` sequences of length N, in place (sequences `npad` elements apart).
// Work item j of a sequence: k = j mod Ns;  v_r = buf[j + r N/R] W^{r k N/(Ns R)};  radix-R butterfly;
// buf[(j / Ns) Ns R + k + r Ns] = v_r.   A thread keeps all its items (at most ITEMS) in registers across the barrier
// that separates the reads of a pass from its writes, so one buffer suffices (half the shared memory of a ping-pong
// scheme: more CTAs per SM).  The twiddles of a pass come from its own table Wq[(r-1) Ns + k] =
// e^{-2 pi i r k / (Ns R)} (conjugated for the inverse): lanes with consecutive k read consecutive entries.
template <int R, int INV>
__device__ __forceinline__ void stockham_pass(cplx *__restrict__ buf, int logN, int Ns, int pairs, int npad,
                                              const double2 *__restrict__ Wq) {
    constexpr int LOGR = R == 8 ? 3 : (R == 4 ? 2 : 1);
    constexpr int ITEMS = 8 / R;                 // 4096 samples and >= 256 threads per CTA: one radix-8 item, two radix-4
    const int logper = logN - LOGR, per = 1 << logper;
    const int total = pairs << logper;
    cplx v[ITEMS][R];
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        const int item = threadIdx.x + it * blockDim.x;
        if (item >= total) continue;
        const int pr = item >> logper, j = item & (per - 1);
        const cplx *s = buf + pr * npad;
        const int k = j & (Ns - 1);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            v[it][r] = s[pad(j + r * per)];
            if (Ns > 1 && r > 0) {
                const double2 w = __ldg(Wq + (r - 1) * Ns + k);
                v[it][r] = cmul(v[it][r], cplx{w.x, INV ? -w.y : w.y});
            }
        }
        if (R == 2) fft2<INV>(v[it]);
        else if (R == 4) fft4<INV>(v[it][0], v[it][1], v[it][2], v[it][3]);
        else fft8<INV>(v[it]);
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        const int item = threadIdx.x + it * blockDim.x;
        if (item >= total) continue;
        const int pr = item >> logper, j = item & (per - 1);
        cplx *d = buf + pr * npad;
        const int k = j & (Ns - 1);
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) d[pad(j0 + r * Ns)] = v[it][r];
    }
    __syncthreads();
}

struct FftParams {
    const double *in;
    double *out;
    const double2 *Wq[4]; // per-pass twiddle tables (see stockham_pass)
    const double2 *T4;    // e^{-i pi k / 2N},   k = 0..N-1
    int N, logN;          // transform length (nx for the x direction, ny for y) = 2^logN
    int bc;               // 0 Neumann, 1 Dirichlet, 2 periodic
    int nx, ny;           // field row length and rows per plane
    int lines;            // x: rows to transform (ny * planes); y: unused
    int blk_in, blk_out;  // y only: that side is the tile-blocked mode-space layout (kernels.cuh); needs nz, k0
    int nz, k0;           // field depth and the z index of the launch's first plane
    int radix[4];         // pass radices (0-terminated)
    double s0, s1;        // forward: output scale of the two special slots / of the others; inverse: input scales
};

// Input position of sample i in the complex sequence, and its sign (Makhoul reordering; DST: alternate signs).
__device__ __forceinline__ int seq_index(int bc, int i, int N, double &sign) {
    sign = 1.0;
    if (bc == 2) return i;
    if (bc == 1 && (i & 1)) sign = -1.0;
    return (i & 1) ? N - 1 - (i >> 1) : (i >> 1);
}
// slots whose basis vector has norm^2 N instead of N/2
__device__ __forceinline__ bool special_slot(int bc, int slot, int N) {
    return bc == 0 ? slot == 0 : (bc == 1 ? slot == N - 1 : (slot == 0 || slot == N - 1));
}

// Line / element addressing, two neighbouring memory elements (one 16-byte access) per step.
// X: a CTA owns `nl` consecutive rows (lines contiguous in memory, N = nx); step e2 -> samples i, i+1 of the two lines
//    l, l+1 of a pair (two 16-byte accesses, two whole complex elements).
// Y: a CTA owns `nl` neighbouring columns of one z-plane (lines strided by nx, N = ny; rows of nl*8 bytes);
//    step e2 -> sample idx of the two lines 2c, 2c+1 — which are exactly the two halves of one complex sequence.
template <bool YP>
struct Lines {
    size_t base;     // element offset of the CTA's first line
    int nl, valid;   // lines of this CTA, and how many of them exist
    int nx, N, logN, lognl;
    __device__ __forceinline__ Lines(const FftParams &p, int nlines, int logn) : nl(nlines), nx(p.nx), N(1 << logn), logN(logn) {
        lognl = 31 - __clz(nlines);
        if (YP) {
            base = (size_t)blockIdx.y * p.nx * p.ny + (size_t)blockIdx.x * nl;
            valid = nl;
        } else {
            const int first = blockIdx.x * nl;
            base = (size_t)first * p.nx;
            valid = min(nl, p.lines - first);
        }
    }
    __device__ __forceinline__ int steps() const { return YP ? (nl << logN) >> 1 : (nl << logN) >> 2; }
    // (first line of a pair, sample index): X steps over two samples of both lines, Y over one sample of both lines
    __device__ __forceinline__ void decode(int e2, int &l, int &idx) const {
        if (YP) { idx = e2 >> (lognl - 1); l = (e2 & ((nl >> 1) - 1)) << 1; }
        else { l = (e2 >> (logN - 1)) << 1; idx = (e2 & ((N >> 1) - 1)) << 1; }
    }
    __device__ __forceinline__ size_t addr(int l, int idx) const { return YP ? base + (size_t)idx * nx + l : base + ((size_t)l << logN) + idx; }
    // y only: mode `idx` of column line l in the tile-blocked layout ((m (nx/16) + i/16) nz + k) 16 + i mod 16
    __device__ __forceinline__ size_t addr_blocked(const FftParams &p, int l, int idx) const {
        const int i = blockIdx.x * nl + l, k = p.k0 + blockIdx.y;
        return (((size_t)idx * (p.nx >> 4) + (i >> 4)) * p.nz + k) * 16 + (i & 15);
    }
};

// Everything that depends only on the transform length is a compile-time constant of the kernel (template LOGN): the
// pass radices, the lines and threads per CTA, every shift, mask and padded offset — index arithmetic was most of the
// instruction count when these were run-time values (profiles/r1d_fft_path.md).
__host__ __device__ constexpr int radix_at(int logn, int q) {            // as many 8s as possible, then 4 (or 4, 4)
    const int n8 = logn / 3, rem = logn % 3;
    if (rem == 1) return q < n8 - 1 ? 8 : (q < n8 + 1 ? 4 : 0);
    return q < n8 ? 8 : ((rem == 2 && q == n8) ? 4 : 0);
}
__host__ __device__ constexpr int lines_of(bool yp, int logn) {          // lines (real sequences) per CTA
    const int n = 1 << logn;
    if (!yp) return n >= 2048 ? 2 : 2 * (2048 / n);                       // x: 4096 samples
    int cols = 8192 / n;                                                  // y: 8192 samples, rows of at least 64 bytes
    if (cols > 16) cols = 16;
    if (cols < 8) cols = n <= 1024 ? 8 : 4;
    return cols;
}
__host__ __device__ constexpr int threads_of(bool yp, int logn) {
    if (!yp) return 256;
    const int t = (lines_of(true, logn) / 2) * ((1 << logn) / 8);
    return t < 64 ? 64 : t;
}
template <int LOGN, int INV, int Q = 0, int NS = 1>
__device__ __forceinline__ void run_passes(cplx *buf, const FftParams &p, int pairs, int npad) {
    constexpr int R = radix_at(LOGN, Q);
    if constexpr (R != 0) {
        stockham_pass<R, INV>(buf, LOGN, NS, pairs, npad, p.Wq[Q]);
        run_passes<LOGN, INV, Q + 1, NS * R>(buf, p, pairs, npad);
    }
}

// spectrum slot -> (FFT bin k, which real combination): value of one line at `slot` from its untangled bin V_k
__device__ __forceinline__ int slot_bin(int bc, int slot, int N) {
    return bc == 2 ? (slot + 1) >> 1 : (bc == 0 ? slot : N - 1 - slot);
}
__device__ __forceinline__ double slot_value(int bc, int slot, cplx V, double2 t4) {
    if (bc == 2) return (slot == 0 || (slot & 1)) ? V.x : -V.y;          // cos rows: Re X_j, sin rows: -Im X_j
    return fma(t4.x, V.x, -t4.y * V.y);                                  // C_k = Re(e^{-i pi k / 2N} V_k)
}

// Forward: out[line][slot] = s(slot) * sum_i q_slot(i) in[line][i]   (Eq. 10 with Q^-1 = Q~^T D^{1/2}, D = w I)
template <bool YP, int LOGN, int BC>
__global__ void __launch_bounds__(threads_of(YP, LOGN), threads_of(YP, LOGN) > 256 ? 2 : 4)
fft_forward_kernel(const FftParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int N = 1 << LOGN, nlines = lines_of(YP, LOGN), pairs = nlines >> 1;
    constexpr int npad = N + (N >> 3) + 1;       // padded length + 1: neighbouring sequences start in different banks
    constexpr int bc = BC;
    cplx *b0 = reinterpret_cast<cplx *>(smem_raw);
    const Lines<YP> L(p, nlines, LOGN);
    const int steps = L.steps();
#pragma unroll 4
    for (int e2 = threadIdx.x; e2 < steps; e2 += blockDim.x) {
        int l, i;
        L.decode(e2, l, i);
        if (YP) {            // v = sample i of lines l, l+1: one complex element
            const double2 v = *reinterpret_cast<const double2 *>(p.in + L.addr(l, i));
            double sign;
            const int n = seq_index(bc, i, N, sign);
            b0[(l >> 1) * npad + pad(n)] = cplx{sign * v.x, sign * v.y};
        } else {             // samples i (even), i+1 of lines l and l+1: two complex elements
            double2 va = make_double2(0.0, 0.0), vb = va;
            if (l < L.valid) va = *reinterpret_cast<const double2 *>(p.in + L.addr(l, i));
            if (l + 1 < L.valid) vb = *reinterpret_cast<const double2 *>(p.in + L.addr(l + 1, i));
            double s0, s1;
            const int n0 = seq_index(bc, i, N, s0), n1 = seq_index(bc, i + 1, N, s1);
            cplx *z = b0 + (l >> 1) * npad;
            z[pad(n0)] = cplx{s0 * va.x, s0 * vb.x};
            z[pad(n1)] = cplx{s1 * va.y, s1 * vb.y};
        }
    }
    __syncthreads();
    run_passes<LOGN, 0>(b0, p, pairs, npad);
    const cplx *Z = b0;
#pragma unroll 4
    for (int e2 = threadIdx.x; e2 < steps; e2 += blockDim.x) {
        int l, slot;
        L.decode(e2, l, slot);
        if (l >= L.valid) continue;
        const cplx *z = Z + (l >> 1) * npad;
        double2 o;
        if (YP) {            // one slot, both lines of the pair
            const int k = slot_bin(bc, slot, N);
            const cplx zk = z[pad(k)], zm = z[pad((N - k) & (N - 1))];
            const double2 t4 = __ldg(p.T4 + k);
            const double sc = special_slot(bc, slot, N) ? p.s0 : p.s1;
            o.x = sc * slot_value(bc, slot, cplx{0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y)}, t4);
            o.y = sc * slot_value(bc, slot, cplx{0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x)}, t4);
        } else {             // slots `slot`, `slot + 1` of both lines of the pair
            double ra[2], rb[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int sl = slot + h, k = slot_bin(bc, sl, N);
                const cplx zk = z[pad(k)], zm = z[pad((N - k) & (N - 1))];
                const double2 t4 = __ldg(p.T4 + k);
                const double sc = special_slot(bc, sl, N) ? p.s0 : p.s1;
                ra[h] = sc * slot_value(bc, sl, cplx{0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y)}, t4);
                rb[h] = sc * slot_value(bc, sl, cplx{0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x)}, t4);
            }
            o = make_double2(ra[0], ra[1]);
            if (l + 1 < L.valid) *reinterpret_cast<double2 *>(p.out + L.addr(l + 1, slot)) = make_double2(rb[0], rb[1]);
        }
        *reinterpret_cast<double2 *>(p.out + ((YP && p.blk_out) ? L.addr_blocked(p, l, slot) : L.addr(l, slot))) = o;
    }
}

// Inverse: out[line][i] = sum_slot q_slot(i) s(slot) in[line][slot]   (Eq. 12 with Q = D^{-1/2} Q~)
template <bool YP, int LOGN, int BC>
__global__ void __launch_bounds__(threads_of(YP, LOGN), threads_of(YP, LOGN) > 256 ? 2 : 4)
fft_inverse_kernel(const FftParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int N = 1 << LOGN, logN = LOGN, nlines = lines_of(YP, LOGN), pairs = nlines >> 1;
    constexpr int npad = N + (N >> 3) + 1;
    constexpr int bc = BC;
    cplx *b0 = reinterpret_cast<cplx *>(smem_raw);
    cplx *Cc = b0;                   // staged scaled coefficients [pair][slot] = (line 2 pr, line 2 pr + 1), overwritten by Z
    constexpr int cstr = N + 1;      // pair stride: neighbouring pairs in different banks
    // (x keeps the two lines of a pair as two real arrays, `rstr` apart: its 16-byte stores are then conflict-free)
    double *Rr = reinterpret_cast<double *>(b0);
    constexpr int rstr = N + 2;
    const Lines<YP> L(p, nlines, LOGN);
    const int steps = L.steps();
#pragma unroll 4
    for (int e2 = threadIdx.x; e2 < steps; e2 += blockDim.x) {
        int l, slot;
        L.decode(e2, l, slot);
        if (YP) {            // slot of lines l, l+1
            const double2 v = *reinterpret_cast<const double2 *>(p.in + (p.blk_in ? L.addr_blocked(p, l, slot) : L.addr(l, slot)));
            const double sc = special_slot(bc, slot, N) ? p.s0 : p.s1;
            Cc[(l >> 1) * cstr + slot] = cplx{sc * v.x, sc * v.y};
        } else {             // slots slot, slot+1 of lines l and l+1
            double2 va = make_double2(0.0, 0.0), vb = va;
            if (l < L.valid) va = *reinterpret_cast<const double2 *>(p.in + L.addr(l, slot));
            if (l + 1 < L.valid) vb = *reinterpret_cast<const double2 *>(p.in + L.addr(l + 1, slot));
            const double sc0 = special_slot(bc, slot, N) ? p.s0 : p.s1, sc1 = special_slot(bc, slot + 1, N) ? p.s0 : p.s1;
            *reinterpret_cast<double2 *>(Rr + l * rstr + slot) = make_double2(sc0 * va.x, sc1 * va.y);
            *reinterpret_cast<double2 *>(Rr + (l + 1) * rstr + slot) = make_double2(sc0 * vb.x, sc1 * vb.y);
        }
    }
    __syncthreads();
    // Hermitian-symmetrised spectrum B of each line (its inverse DFT is real); the pair rides as Z = B_even + i B_odd.
    // Built in registers (at most ZITEMS elements per thread), then written over the staged coefficients.
    constexpr int ZITEMS = 8;
    cplx zreg[ZITEMS];
#pragma unroll
    for (int it = 0; it < ZITEMS; ++it) {
        const int item = threadIdx.x + it * blockDim.x;
        if (item >= (pairs << logN)) continue;
        const int pr = item >> logN, k = item & (N - 1);
        cplx B[2];
        // scaled coefficient q of both lines of the pair
        auto c = [&](int q) -> cplx {
            if (YP) return Cc[pr * cstr + q];
            return cplx{Rr[2 * pr * rstr + q], Rr[(2 * pr + 1) * rstr + q]};
        };
        if (bc == 2) {
            const int j = k <= N / 2 ? k : N - k;                          // B_k = b_k / 2, B_{N-k} = conj(b_k) / 2
            if (j == 0 || j == N / 2) {
                const cplx a = c(j == 0 ? 0 : N - 1);
                B[0] = {a.x, 0.0};
                B[1] = {a.y, 0.0};
            } else {
                const cplx ar = c(2 * j - 1), ai = c(2 * j);
                const double sg = k < N / 2 ? -0.5 : 0.5;
                B[0] = {0.5 * ar.x, sg * ai.x};
                B[1] = {0.5 * ar.y, sg * ai.y};
            }
        } else if (k == 0) {
            const cplx a = c(bc == 0 ? 0 : N - 1);
            B[0] = {a.x, 0.0};
            B[1] = {a.y, 0.0};
        } else {
            const cplx ak = c(bc == 0 ? k : N - 1 - k), am = c(bc == 0 ? N - k : k - 1);
            const double2 t = __ldg(p.T4 + k);                             // e^{+i pi k / 2N} (a_k - i a_{N-k}) / 2
            B[0] = cmul(cplx{0.5 * t.x, -0.5 * t.y}, cplx{ak.x, -am.x});
            B[1] = cmul(cplx{0.5 * t.x, -0.5 * t.y}, cplx{ak.y, -am.y});
        }
        zreg[it] = cplx{B[0].x - B[1].y, B[0].y + B[1].x};
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < ZITEMS; ++it) {
        const int item = threadIdx.x + it * blockDim.x;
        if (item >= (pairs << logN)) continue;
        b0[(item >> logN) * npad + pad(item & (N - 1))] = zreg[it];
    }
    __syncthreads();
    run_passes<LOGN, 1>(b0, p, pairs, npad);
    const cplx *Z = b0;
#pragma unroll 4
    for (int e2 = threadIdx.x; e2 < steps; e2 += blockDim.x) {
        int l, i;
        L.decode(e2, l, i);
        if (l >= L.valid) continue;
        const cplx *z = Z + (l >> 1) * npad;
        double2 o;
        if (YP) {
            double sign;
            const cplx c = z[pad(seq_index(bc, i, N, sign))];
            o = make_double2(sign * c.x, sign * c.y);
        } else {
            double s0, s1;
            const cplx c0 = z[pad(seq_index(bc, i, N, s0))], c1 = z[pad(seq_index(bc, i + 1, N, s1))];
            o = make_double2(s0 * c0.x, s1 * c1.x);              // line l: real parts; line l + 1: imaginary parts
            if (l + 1 < L.valid) *reinterpret_cast<double2 *>(p.out + L.addr(l + 1, i)) = make_double2(s0 * c0.y, s1 * c1.y);
        }
        *reinterpret_cast<double2 *>(p.out + L.addr(l, i)) = o;
    }
}

}  // namespace

// pass radices of a length-2^m transform: as many 8s as possible, then 4 (or 4, 4); at most 4 passes for n <= 2048
static int fft_radices(int n, int radix[4]) {
    int m = 0;
    while ((1 << m) < n) ++m;
    int q = 0;
    const int n8 = m / 3, rem = m % 3;
    radix[0] = radix[1] = radix[2] = radix[3] = 0;
    if (rem == 1) {
        for (int r = 0; r < n8 - 1; ++r) radix[q++] = 8;
        radix[q++] = 4; radix[q++] = 4;
    } else {
        for (int r = 0; r < n8; ++r) radix[q++] = 8;
        if (rem == 2) radix[q++] = 4;
    }
    return m;
}

bool fft_supported(int n) { return n >= 16 && n <= 2048 && (n & (n - 1)) == 0; }

// Host side of the twiddle tables, interleaved (re, im): T4[k] = e^{-i pi k / 2N} (n entries), then for every pass
// after the first its table e^{-2 pi i r k / (Ns R)}, r = 1..R-1, k = 0..Ns-1.
void fft_tables(int n, std::vector<double> &out) {
    const long double pi = 3.14159265358979323846264338327950288L;
    out.clear();
    for (int t = 0; t < n; ++t) {
        const long double b = -pi * t / (2.0L * n);
        out.push_back((double)cosl(b));
        out.push_back((double)sinl(b));
    }
    int radix[4];
    fft_radices(n, radix);
    int Ns = 1;
    for (int q = 0; q < 4 && radix[q]; ++q) {
        const int R = radix[q];
        if (q > 0)
            for (int r = 1; r < R; ++r)
                for (int k = 0; k < Ns; ++k) {
                    const long double a = -2.0L * pi * r * k / ((long double)Ns * R);
                    out.push_back((double)cosl(a));
                    out.push_back((double)sinl(a));
                }
        Ns *= R;
    }
}

cudaError_t fft_configure() { return cudaSuccess; }   // shared-memory opt-in happens per instantiation at first launch

namespace {

template <bool YP, int LOGN, int BC>
cudaError_t launch_bc(const FftParams &p, int inverse, int grid_x, int grid_y, cudaStream_t stream) {
    constexpr int N = 1 << LOGN, nl = lines_of(YP, LOGN), threads = threads_of(YP, LOGN);
    constexpr size_t smem = (size_t)(nl / 2) * (N + (N >> 3) + 1) * 16;
    if (smem > 48 * 1024) {
        static DeviceOnce configured;                        // per device, thread-safe (devonce.hpp)
        cudaError_t e = configured.run([&] {
            cudaError_t q = cudaFuncSetAttribute(fft_forward_kernel<YP, LOGN, BC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (q == cudaSuccess) q = cudaFuncSetAttribute(fft_inverse_kernel<YP, LOGN, BC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            return q;
        });
        if (e != cudaSuccess) return e;
    }
    const dim3 grid(grid_x, grid_y);
    if (inverse) fft_inverse_kernel<YP, LOGN, BC><<<grid, threads, smem, stream>>>(p);
    else fft_forward_kernel<YP, LOGN, BC><<<grid, threads, smem, stream>>>(p);
    return cudaGetLastError();
}

template <bool YP, int LOGN>
cudaError_t launch_one(const FftParams &p, int inverse, int grid_x, int grid_y, cudaStream_t stream) {
    if (p.bc == 0) return launch_bc<YP, LOGN, 0>(p, inverse, grid_x, grid_y, stream);
    if (p.bc == 1) return launch_bc<YP, LOGN, 1>(p, inverse, grid_x, grid_y, stream);
    return launch_bc<YP, LOGN, 2>(p, inverse, grid_x, grid_y, stream);
}

template <bool YP>
cudaError_t launch_len(const FftParams &p, int inverse, int grid_x, int grid_y, cudaStream_t stream) {
    switch (p.logN) {
        case 4: return launch_one<YP, 4>(p, inverse, grid_x, grid_y, stream);
        case 5: return launch_one<YP, 5>(p, inverse, grid_x, grid_y, stream);
        case 6: return launch_one<YP, 6>(p, inverse, grid_x, grid_y, stream);
        case 7: return launch_one<YP, 7>(p, inverse, grid_x, grid_y, stream);
        case 8: return launch_one<YP, 8>(p, inverse, grid_x, grid_y, stream);
        case 9: return launch_one<YP, 9>(p, inverse, grid_x, grid_y, stream);
        case 10: return launch_one<YP, 10>(p, inverse, grid_x, grid_y, stream);
        case 11: return launch_one<YP, 11>(p, inverse, grid_x, grid_y, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t launch_fft(const FftArgs &a, cudaStream_t stream) {
    const int N = a.dir == 0 ? a.nx : a.ny;
    if (!fft_supported(N) || a.planes < 1) return cudaErrorInvalidValue;
    FftParams p{};
    p.in = a.in; p.out = a.out;
    p.T4 = reinterpret_cast<const double2 *>(a.tables);
    p.N = N; p.bc = a.bc; p.nx = a.nx; p.ny = a.ny;
    p.s0 = a.s0; p.s1 = a.s1;
    p.blk_in = a.dir == 1 && a.inverse && a.blocked; p.blk_out = a.dir == 1 && !a.inverse && a.blocked;
    p.nz = a.nz; p.k0 = a.k0;
    p.logN = fft_radices(N, p.radix);
    {
        const double2 *w = p.T4 + N;
        int Ns = 1;
        for (int q = 0; q < 4 && p.radix[q]; ++q) {
            p.Wq[q] = w;
            if (q > 0) w += (p.radix[q] - 1) * Ns;
            Ns *= p.radix[q];
        }
    }
    if (a.dir == 0) {
        const int nl = lines_of(false, p.logN);
        p.lines = a.ny * a.planes;
        return launch_len<false>(p, a.inverse, (p.lines + nl - 1) / nl, 1, stream);
    }
    const int cols = lines_of(true, p.logN);
    if (a.nx % cols) return cudaErrorInvalidValue;
    return launch_len<true>(p, a.inverse, a.nx / cols, a.planes, stream);
}

}  // namespace tpt
