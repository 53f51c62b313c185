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

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;\n" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory"); }   // see ptx.cuh

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
// Radix-16 passes (N >= 1024) store with stride 16 (forward, first pass) and in blocks of 4 every 64 (inverse, second pass):
// the forward transform then pads one element per 16, the inverse adds half a bank round per 64 (profiles: 26-30 % of the
// shared-memory wavefronts of the 1024-long transforms were conflict replays with the plain padding).
template <int LOGN, int INV>
__device__ __forceinline__ int padf(int i) {
    if (LOGN < 10) return i + (i >> 3);
    return INV ? i + (i >> 3) + 4 * (i >> 6) : i + (i >> 4);
}

struct FftParams {
    const double *in;
    double *out;
    const double2 *Wq[4]; // per-pass twiddle tables: Wq[q][(r-1) Ns + k] = e^{-2 pi i r k / (Ns R)}
    const double2 *T4;    // e^{-i pi k / 2N},   k = 0..N-1
    int N, logN;          // transform length (nx for the x direction, ny for y) = 2^logN
    int bc;               // 0 Neumann, 1 Dirichlet, 2 periodic
    int nx, ny;           // field row length and rows per plane
    int lines;            // x: rows to transform (ny * planes)
    int planes;           // y: z-planes of this launch
    int blk_in, blk_out;  // y only: that side is the tile-blocked mode-space layout (kernels.cuh); needs nz, k0
    int nz, k0;           // field depth and the z index of the launch's first plane
    int bgroups;          // y only: 16-column groups per mode row of the blocked side (nx/16, or the slab width / 16)
    int radix[4];         // pass radices (0-terminated)
    double s0, s1;        // forward: output scale of the two special slots / of the others; inverse: input scales
    int npeers, units;    // sharded forward y: owner of mode row m = ((m >> 4) + 1) npeers - 1) / units, stored through peer_out
    double *peer_out[MAX_PEERS];
};

// Everything that depends only on the transform length is a compile-time constant of the kernel (template LOGN): the
// pass radices, the lines per CTA, every shift, mask and padded offset.
// Pass radices.  Up to N = 512: as many 8s as possible, then 4 (or 4, 4) — at most three passes.  N = 1024 / 2048 would need
// four radix-8/4 passes = three exchanges through shared memory, the pipe these kernels saturate first; with radix-16
// passes (one item of 16 values per thread) they need three: 16, 16, 4 / 16, 16, 8.  The pass that works on conjugate-paired
// items (last forward, first inverse) needs two items per thread, i.e. radix 4 or 8: the inverse runs the same radices
// in the opposite order (4, 16, 16 / 8, 16, 16) with its own twiddle tables.
__host__ __device__ constexpr int radix_at(int logn, int q, int inv = 0) {
    if (logn >= 10) {
        const int small = logn == 10 ? 4 : 8;
        if (q > 2) return 0;
        return inv ? (q == 0 ? small : 16) : (q == 2 ? small : 16);
    }
    const int n8 = logn / 3, rem = logn % 3;
    if (rem == 1) return q < n8 - 1 ? 8 : (q < n8 + 1 ? 4 : 0);
    return q < n8 ? 8 : ((rem == 2 && q == n8) ? 4 : 0);
}
__host__ __device__ constexpr int npasses(int logn) { return radix_at(logn, 1) == 0 ? 1 : (radix_at(logn, 2) == 0 ? 2 : (radix_at(logn, 3) == 0 ? 3 : 4)); }

// Geometry of one CTA: every thread holds 16 complex values (two real lines ride in one complex sequence).
//   x: 4096 / N consecutive rows, 128 threads (four CTAs per SM interleave their load / compute / store phases).
//   y: 8192 samples, 256 threads: a tile of COLS neighbouring columns (128-byte rows up to N = 512, 64 / 32 bytes
//   for N = 1024 / 2048) of PL consecutive z-planes.
// Thread t holds the 16 values of its work items in registers through every pass.  Thread <-> (pair of lines pr, slice u
// of the sequence, u in [0, N/16)):  y: pr fastest — the 8 lanes of a quarter-warp are the 8 column pairs of one row, so
// every global access is a whole 128-byte row and every shared-memory access hits 8 different sequences (NPAD keeps
// them in different banks);  x: u fastest — consecutive lanes hold consecutive sequence elements.
template <bool YP, int LOGN>
struct Geo {
    static constexpr int N = 1 << LOGN;
    static constexpr int COLS = N <= 512 ? 16 : (N == 1024 ? 8 : 4);
    static constexpr int PL = N >= 512 ? 1 : 512 / N;
    static constexpr int LINES = YP ? COLS * PL : (N >= 2048 ? 2 : 4096 / N);
    static constexpr int PAIRS = LINES / 2;
    static constexpr int UPP = N / 16;
    static constexpr int THREADS = PAIRS * UPP;                          // y: 256, x: 128
    static constexpr int MINB = 512 / THREADS;                           // CTAs per SM the 128-register budget admits
    static constexpr int BANKSTEP = !YP ? 1 : (COLS == 16 ? 1 : (COLS == 8 ? 2 : 4));
    static constexpr int NPAD = ((N + (N >> 3) + (N >= 1024 ? (N >> 4) : 0) + 7) & ~7) + BANKSTEP;   // padded sequence length (complex elements; covers padf)
    static constexpr size_t SMEM = (size_t)PAIRS * NPAD * 16;
};

// 16-point DFT in registers as 4 x 4: radix-4 over the stride-4 subsets, twiddles W16^{a b}, radix-4 across; the result
// of frequency b + 4c lands in slot 4b + c and is renamed into natural order.
template <int INV>
__device__ __forceinline__ void fft16(cplx *v) {
    constexpr double c1 = 0.92387953251128675613, s1 = 0.38268343236508977173, h = 0.70710678118654752440;
#pragma unroll
    for (int a = 0; a < 4; ++a) fft4<INV>(v[a], v[a + 4], v[a + 8], v[a + 12]);      // v[a + 4b] = sum_m x[a + 4m] W4^{m b}
    auto tw = [&](cplx &z, double wr, double wi) { z = cmul(z, cplx{wr, INV ? -wi : wi}); };   // W16^q = (wr, wi), forward sign
    tw(v[1 + 4], c1, -s1);  tw(v[2 + 4], h, -h);     tw(v[3 + 4], s1, -c1);          // b = 1: q = 1, 2, 3
    tw(v[1 + 8], h, -h);    v[2 + 8] = mul_mi<INV>(v[2 + 8]);  tw(v[3 + 8], -h, -h); // b = 2: q = 2, 4, 6
    tw(v[1 + 12], s1, -c1); tw(v[2 + 12], -h, -h);   tw(v[3 + 12], -c1, s1);         // b = 3: q = 3, 6, 9
#pragma unroll
    for (int b = 0; b < 4; ++b) fft4<INV>(v[4 * b], v[4 * b + 1], v[4 * b + 2], v[4 * b + 3]);   // v[4b + c] = X[b + 4c]
    cplx t[16];
#pragma unroll
    for (int b = 0; b < 4; ++b)
#pragma unroll
        for (int c = 0; c < 4; ++c) t[b + 4 * c] = v[4 * b + c];
#pragma unroll
    for (int q = 0; q < 16; ++q) v[q] = t[q];
}

template <int R, int INV>
__device__ __forceinline__ void bfly(cplx *v) {
    if (R == 16) fft16<INV>(v);
    else if (R == 8) fft8<INV>(v);
    else fft4<INV>(v[0], v[1], v[2], v[3]);
}
// v_r *= W^{r k}, W = e^{-+2 pi i / (Ns R)}, from the pass table Wq[(r-1) Ns + k].  DERIVE: load only W^k, W^2k (and W^4k) and
// form the other powers by complex multiplication — in the x kernels consecutive lanes hold consecutive k, so every
// table load is a full 512-byte warp access and seven of them per item cost more L1 bandwidth than the data itself.
template <int R, int INV, bool DERIVE>
__device__ __forceinline__ void twiddle(cplx *v, const double2 *__restrict__ Wq, int Ns, int k) {
    if (!DERIVE) {
#pragma unroll
        for (int r = 1; r < R; ++r) {
            const double2 w = __ldg(Wq + (r - 1) * Ns + k);
            v[r] = cmul(v[r], cplx{w.x, INV ? -w.y : w.y});
        }
    } else {
        const double2 a = __ldg(Wq + k), b = __ldg(Wq + Ns + k);
        const cplx w1{a.x, INV ? -a.y : a.y}, w2{b.x, INV ? -b.y : b.y};
        const cplx w3 = cmul(w1, w2);
        v[1] = cmul(v[1], w1);
        v[2] = cmul(v[2], w2);
        v[3] = cmul(v[3], w3);
        if (R >= 8) {
            const double2 c = __ldg(Wq + 3 * Ns + k);
            const cplx w4{c.x, INV ? -c.y : c.y};
            const cplx w5 = cmul(w4, w1), w6 = cmul(w4, w2), w7 = cmul(w4, w3);
            v[4] = cmul(v[4], w4);
            v[5] = cmul(v[5], w5);
            v[6] = cmul(v[6], w6);
            v[7] = cmul(v[7], w7);
            if (R == 16) {
                const double2 d = __ldg(Wq + 7 * Ns + k);
                const cplx w8{d.x, INV ? -d.y : d.y};
                v[8] = cmul(v[8], w8);
                v[9] = cmul(v[9], cmul(w8, w1));
                v[10] = cmul(v[10], cmul(w8, w2));
                v[11] = cmul(v[11], cmul(w8, w3));
                v[12] = cmul(v[12], cmul(w8, w4));
                v[13] = cmul(v[13], cmul(w8, w5));
                v[14] = cmul(v[14], cmul(w8, w6));
                v[15] = cmul(v[15], cmul(w8, w7));
            }
        }
    }
}

// Sample position of element n of the complex sequence, and its sign (Makhoul reordering v_n = f_{2n},
// v_{N-1-n} = f_{2n+1}; the sine transform alternates signs; the periodic case is the plain DFT).
template <int BC, int N>
__device__ __forceinline__ int sample_of(int n, double &sign) {
    sign = 1.0;
    if (BC == 2) return n;
    const int i = n < N / 2 ? 2 * n : 2 * (N - 1 - n) + 1;
    if (BC == 1 && (i & 1)) sign = -1.0;
    return i;
}
// slots whose basis vector has norm^2 N instead of N/2
template <int BC, int N>
__device__ __forceinline__ bool special_slot(int slot) {
    return BC == 0 ? slot == 0 : (BC == 1 ? slot == N - 1 : (slot == 0 || slot == N - 1));
}

// Middle passes Q = 1 .. NP-2: in-place Stockham pass through shared memory.  Item j of a sequence: k = j mod Ns;
// v_r = buf[j + r N/R] W^{r k}; radix-R butterfly; buf[(j - k) R + k + r Ns] = v_r.
template <int LOGN, int INV, int Q, int NS, int UPP, bool XDIR>
__device__ __forceinline__ void middle_passes(cplx *seq, cplx *v, const FftParams &p, int u) {
    constexpr int NP = npasses(LOGN), N = 1 << LOGN;
    if constexpr (Q < NP - 1) {
        constexpr int R = radix_at(LOGN, Q, INV), IT = 16 / R, PER = N / R;
#pragma unroll
        for (int it = 0; it < IT; ++it) {
            const int j = u + it * UPP, k = j & (NS - 1);
#pragma unroll
            for (int r = 0; r < R; ++r) v[it * R + r] = seq[padf<LOGN, INV>(j + r * PER)];
            twiddle<R, INV, (XDIR && NS >= 32)>(v + it * R, p.Wq[Q], NS, k);
            bfly<R, INV>(v + it * R);
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < IT; ++it) {
            const int j = u + it * UPP, k = j & (NS - 1);
#pragma unroll
            for (int r = 0; r < R; ++r) seq[padf<LOGN, INV>((j - k) * R + k + r * NS)] = v[it * R + r];
        }
        __syncthreads();
        middle_passes<LOGN, INV, Q + 1, NS * R, UPP, XDIR>(seq, v, p, u);
    }
}
// e^{-i pi r / (2 R)}: T4[j + r N/R] = T4[j] * rot<R>(r), so the post-/pre-twiddles e^{-i pi k / 2N} of all bins of an item
// follow from ONE table entry (and T4[N - k] = -i conj T4[k] needs none): 2 table loads per thread instead of 16.
template <int R>
__device__ __forceinline__ cplx rot(int r) {
    constexpr double c1 = 0.98078528040323044913, s1 = 0.19509032201612826785;   // pi/16
    constexpr double c2 = 0.92387953251128675613, s2 = 0.38268343236508977173;   // pi/8
    constexpr double c3 = 0.83146961230254523708, s3 = 0.55557023301960222474;   // 3 pi/16
    constexpr double c4 = 0.70710678118654752440;                                // pi/4
    const int q = R == 8 ? r : 2 * r;                                            // angle = q pi / 16
    switch (q) {
        case 0: return cplx{1.0, 0.0};
        case 1: return cplx{c1, -s1};
        case 2: return cplx{c2, -s2};
        case 3: return cplx{c3, -s3};
        case 4: return cplx{c4, -c4};
        case 5: return cplx{s3, -c3};
        case 6: return cplx{s2, -c2};
        default: return cplx{s1, -c1};
    }
}
// e^{-i pi / (4 R)}: T4[N / (2R)], the first bin of the self-paired item PER/2
template <int R>
__device__ __forceinline__ cplx rot_half() {
    return R == 8 ? cplx{0.99518472667219688624, -0.09801714032956060199} : cplx{0.98078528040323044913, -0.19509032201612826785};
}

// Items of the pass whose bins must come in conjugate pairs (k, N - k) — the last forward pass (untangling the two
// real lines needs Z_k and Z_{N-k}) and the first inverse pass (a Hermitian spectrum is built from a_k and a_{N-k}).
// Item j covers the bins j + r PER (PER = N/R); the partner bins N - j - r PER belong to item PER - j, r' = R-1-r.  A
// thread therefore takes the items (u, PER - u) [and (u + UPP, PER - UPP - u) for radix 4]; the self-paired items 0 and
// PER/2 go together to thread u = 0.
template <int R, int PER, int UPP>
__device__ __forceinline__ void paired_items(int u, int *j) {
    j[0] = u;
    j[1] = u ? PER - u : PER / 2;
    if (R == 4) {
        j[2] = u + UPP;
        j[3] = PER - UPP - u;
    }
}

// ---- per-CTA line addressing --------------------------------------------------------------------------------------
// y: row idx of my column pair (both lines: one 16-byte access) lives at base + idx * stride on either side — natural
//    layout: stride nx; tile-blocked layout ((idx bgroups + col/16) nz + k) 16 + col%16: stride bgroups * nz * 16.
// x: my two lines are rows of N contiguous elements.
template <bool YP, int LOGN>
struct Addr {
    using G = Geo<YP, LOGN>;
    size_t in_base, out_base, in_stride, out_stride;
    bool ok0, ok1;        // the two lines of my pair exist
    __device__ __forceinline__ Addr(const FftParams &p, int pr) {
        if (YP) {
            const int cp = pr % (G::COLS / 2), pl = pr / (G::COLS / 2);
            const int col = blockIdx.x * G::COLS + 2 * cp;
            const int plane = blockIdx.y * G::PL + pl;
            ok0 = ok1 = plane < p.planes;
            const size_t nat = (size_t)plane * p.nx * p.ny + col;
            const size_t blk = ((size_t)(col >> 4) * p.nz + (p.k0 + plane)) * 16 + (col & 15);
            const size_t bstride = (size_t)p.bgroups * p.nz * 16;
            in_base = p.blk_in ? blk : nat;
            in_stride = p.blk_in ? bstride : (size_t)p.nx;
            out_base = p.blk_out ? blk : nat;
            out_stride = p.blk_out ? bstride : (size_t)p.nx;
        } else {
            const int l = blockIdx.x * G::LINES + 2 * pr;
            ok0 = l < p.lines;
            ok1 = l + 1 < p.lines;
            in_base = out_base = (size_t)l << LOGN;
            in_stride = out_stride = 0;
        }
    }
};

// Forward: out[line][slot] = s(slot) * sum_i q_slot(i) in[line][i]   (Eq. 10 with Q^-1 = Q~^T D^{1/2}, D = w I)
//   y: the first pass reads its 16 rows straight from global memory (whole 128-byte rows per quarter-warp);
//   x: the rows are staged once through shared memory (coalesced 16-byte loads, Makhoul scatter);
//   last pass: paired items, the two lines untangled in registers, every result stored straight to global memory.
// PEERS (y only): the sharded solve's exchange 1 — every mode row is stored through the base pointer of its owner.
template <bool YP, int LOGN, int BC, bool PEERS = false>
__global__ void __launch_bounds__(Geo<YP, LOGN>::THREADS, Geo<YP, LOGN>::MINB) fft_forward_kernel(const FftParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using G = Geo<YP, LOGN>;
    constexpr int N = G::N, NP = npasses(LOGN), UPP = G::UPP, NPAD = G::NPAD;
    cplx *buf = reinterpret_cast<cplx *>(smem_raw);
    const int t = threadIdx.x;
    const int pr = YP ? t % G::PAIRS : t / UPP;
    const int u = YP ? t / G::PAIRS : t % UPP;
    cplx *seq = buf + pr * NPAD;
    const Addr<YP, LOGN> A(p, pr);
    cplx v[16];
    pdl_launch_dependents();
    pdl_wait();                   // the input is the previous kernel's output

    // ---- pass 0 (Ns = 1: no twiddles) -------------------------------------------------------------------------------
    constexpr int R0 = radix_at(LOGN, 0), IT0 = 16 / R0, PER0 = N / R0;
    if (YP) {
        // all 16 loads are issued before the first use (no branch, no arithmetic on a loaded value in between)
        if (A.ok0) {
            const double *src = p.in + A.in_base;
#pragma unroll
            for (int it = 0; it < IT0; ++it)
#pragma unroll
                for (int r = 0; r < R0; ++r) {
                    double sg;
                    const int i = sample_of<BC, N>(u + it * UPP + r * PER0, sg);
                    const double2 w = *reinterpret_cast<const double2 *>(src + (size_t)i * A.in_stride);
                    v[it * R0 + r] = cplx{w.x, w.y};
                }
        } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) v[q] = cplx{0.0, 0.0};
        }
        if (BC == 1) {
#pragma unroll
            for (int it = 0; it < IT0; ++it)
#pragma unroll
                for (int r = 0; r < R0; ++r) {
                    double sg;
                    sample_of<BC, N>(u + it * UPP + r * PER0, sg);
                    v[it * R0 + r] = cplx{sg * v[it * R0 + r].x, sg * v[it * R0 + r].y};
                }
        }
    } else {
        // x: sample i(n) of both lines straight into registers.  Makhoul's order makes these 8-byte loads stride-2 across the
        // lanes (even samples ascending for the first half of the sequence, odd samples descending for the second); the
        // other half of every 32-byte sector is asked for by the mirrored lane of the same warp a few instructions later
        // (an L1 hit), which costs less L1 bandwidth than staging the rows through shared memory (one store + one load
        // per element and two barriers more).
        if (A.ok0) {
            const double *src0 = p.in + A.in_base;
            const double *src1 = A.ok1 ? src0 + N : src0;
#pragma unroll
            for (int it = 0; it < IT0; ++it)
#pragma unroll
                for (int r = 0; r < R0; ++r) {
                    double sg;
                    const int i = sample_of<BC, N>(u + it * UPP + r * PER0, sg);
                    v[it * R0 + r] = cplx{src0[i], src1[i]};
                }
            if (!A.ok1) {
#pragma unroll
                for (int q = 0; q < 16; ++q) v[q].y = 0.0;
            }
        } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) v[q] = cplx{0.0, 0.0};
        }
        if (BC == 1) {
#pragma unroll
            for (int it = 0; it < IT0; ++it)
#pragma unroll
                for (int r = 0; r < R0; ++r) {
                    double sg;
                    sample_of<BC, N>(u + it * UPP + r * PER0, sg);
                    v[it * R0 + r] = cplx{sg * v[it * R0 + r].x, sg * v[it * R0 + r].y};
                }
        }
    }
#pragma unroll
    for (int it = 0; it < IT0; ++it) {
        bfly<R0, 0>(v + it * R0);
#pragma unroll
        for (int r = 0; r < R0; ++r) seq[padf<LOGN, 0>((u + it * UPP) * R0 + r)] = v[it * R0 + r];
    }
    __syncthreads();
    middle_passes<LOGN, 0, 1, R0, UPP, !YP>(seq, v, p, u);

    // ---- last pass: paired items; Ns = PER = N / R ---------------------------------------------------------------------
    constexpr int RL = radix_at(LOGN, NP - 1), ITL = 16 / RL, NSL = N / RL;
    int jl[4];
    paired_items<RL, NSL, UPP>(u, jl);
    cplx tb0{1.0, 0.0}, tb2{1.0, 0.0};                       // e^{-i pi j / 2N} of my items (BC 0 / 1); latency hides under the pass
    if (BC != 2) {
        const double2 w0 = __ldg(p.T4 + jl[0]);
        tb0 = cplx{w0.x, w0.y};
        if (RL == 4) {
            const double2 w2 = __ldg(p.T4 + jl[2]);
            tb2 = cplx{w2.x, w2.y};
        }
    }
#pragma unroll
    for (int it = 0; it < ITL; ++it) {
#pragma unroll
        for (int r = 0; r < RL; ++r) v[it * RL + r] = seq[padf<LOGN, 0>(jl[it] + r * NSL)];
        twiddle<RL, 0, (!YP && NSL >= 32)>(v + it * RL, p.Wq[NP - 1], NSL, jl[it]);
        bfly<RL, 0>(v + it * RL);
    }
    // v[it RL + r] = Z[jl[it] + r NSL].  Untangle (V1_k = (Z_k + conj Z_{N-k}) / 2, V2_k = (Z_k - conj Z_{N-k}) / 2i;
    // V_{N-k} = conj V_k for real lines), apply e^{-i pi k / 2N}, scale, store.
    auto store = [&](int slot, double o1, double o2) {
        const double sc = special_slot<BC, N>(slot) ? p.s0 : p.s1;
        if (YP) {
            // sharded solve: the owner of mode row `slot` receives it straight from this store (exchange 1 of sharded.cu)
            double *dst = PEERS ? p.peer_out[(((slot >> 4) + 1) * p.npeers - 1) / p.units] : p.out;
            if (A.ok0) *reinterpret_cast<double2 *>(dst + A.out_base + (size_t)slot * A.out_stride) = make_double2(sc * o1, sc * o2);
        } else {
            if (A.ok0) p.out[A.out_base + slot] = sc * o1;
            if (A.ok1) p.out[A.out_base + N + slot] = sc * o2;
        }
    };
    // bins k and N - k; zm = Z_{N-k}; tk = e^{-i pi k / 2N};  0 < k < N, k != N/2
    auto emit = [&](int k, cplx tk, cplx zk, cplx zm) {
        const cplx V1{0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y)}, V2{0.5 * (zk.y + zm.y), 0.5 * (zm.x - zk.x)};
        if (BC == 2) {
            const int kk = k < N / 2 ? k : N - k;
            const double sg = k < N / 2 ? -1.0 : 1.0;           // slot 2kk-1: Re V_kk, slot 2kk: -Im V_kk
            store(2 * kk - 1, V1.x, V2.x);
            store(2 * kk, sg * V1.y, sg * V2.y);
        } else {
            const cplx tm{-tk.y, -tk.x};                         // e^{-i pi (N-k) / 2N} = -i conj tk
            store(BC == 0 ? k : N - 1 - k, fma(tk.x, V1.x, -tk.y * V1.y), fma(tk.x, V2.x, -tk.y * V2.y));
            store(BC == 0 ? N - k : k - 1, fma(tm.x, V1.x, tm.y * V1.y), fma(tm.x, V2.x, tm.y * V2.y));
        }
    };
    auto emit_single = [&](int k, cplx z) {                  // k = 0 or N/2: its own partner; V1 = Re Z, V2 = Im Z
        if (BC == 2) {
            store(k == 0 ? 0 : N - 1, z.x, z.y);
        } else {
            const double tx = k == 0 ? 1.0 : 0.70710678118654752440;    // Re e^{-i pi k / 2N}
            store(BC == 0 ? k : N - 1 - k, tx * z.x, tx * z.y);
        }
    };
    if (RL == 4) {
#pragma unroll
        for (int r = 0; r < RL; ++r) emit(jl[2] + r * NSL, cmul(tb2, rot<RL>(r)), v[2 * RL + r], v[3 * RL + RL - 1 - r]);
    }
    if (u) {
#pragma unroll
        for (int r = 0; r < RL; ++r) emit(jl[0] + r * NSL, cmul(tb0, rot<RL>(r)), v[r], v[RL + RL - 1 - r]);
    } else {
        emit_single(0, v[0]);
        emit_single(N / 2, v[RL / 2]);
#pragma unroll
        for (int r = 1; r < RL / 2; ++r) emit(r * NSL, rot<RL>(r), v[r], v[RL - r]);
#pragma unroll
        for (int r = 0; r < RL / 2; ++r) emit(NSL / 2 + r * NSL, cmul(rot_half<RL>(), rot<RL>(r)), v[RL + r], v[RL + RL - 1 - r]);
    }
}

// Inverse: out[line][i] = sum_slot q_slot(i) s(slot) in[line][slot]   (Eq. 12 with Q = D^{-1/2} Q~)
//   first pass: paired items; the Hermitian-symmetrised spectrum B of each line (its inverse DFT is real; the pair rides
//   as Z = B_1 + i B_2) is built in registers straight from the global loads of the scaled coefficients;
//   y: the last pass stores its 16 rows straight to global memory;  x: one pass through shared memory for coalesced rows.
template <bool YP, int LOGN, int BC>
__global__ void __launch_bounds__(Geo<YP, LOGN>::THREADS, Geo<YP, LOGN>::MINB) fft_inverse_kernel(const FftParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using G = Geo<YP, LOGN>;
    constexpr int N = G::N, NP = npasses(LOGN), UPP = G::UPP, NPAD = G::NPAD;
    cplx *buf = reinterpret_cast<cplx *>(smem_raw);
    const int t = threadIdx.x;
    const int pr = YP ? t % G::PAIRS : t / UPP;
    const int u = YP ? t / G::PAIRS : t % UPP;
    cplx *seq = buf + pr * NPAD;
    const Addr<YP, LOGN> A(p, pr);
    cplx v[16];
    pdl_launch_dependents();
    pdl_wait();                   // the input is the previous kernel's output

    // ---- first pass: paired items, inputs built from the coefficients ---------------------------------------------------
    constexpr int R0 = radix_at(LOGN, 0, 1), IT0 = 16 / R0, PER0 = N / R0;
    int j0[4];
    paired_items<R0, PER0, UPP>(u, j0);
    // Every register position first receives the coefficient its own bin contributes: bin k of a cosine / sine transform
    // the coefficient a_k; of the real DFT, a bin below N/2 the cosine coefficient of its frequency and its partner N - k
    // the sine coefficient.  All 16 loads are issued before the first use (no branch, no arithmetic in between); the
    // scales follow, then the conjugate pairs are combined in place.
    auto slot_for = [&](int k) -> int {
        if (BC == 0) return k;
        if (BC == 1) return N - 1 - k;
        return k == 0 ? 0 : (k == N / 2 ? N - 1 : (k < N / 2 ? 2 * k - 1 : 2 * (N - k)));
    };
    cplx tb0{1.0, 0.0}, tb2{1.0, 0.0};                       // e^{-i pi j / 2N} of my items (BC 0 / 1)
    if (BC != 2) {
        const double2 w0 = __ldg(p.T4 + j0[0]);
        tb0 = cplx{w0.x, w0.y};
        if (R0 == 4) {
            const double2 w2 = __ldg(p.T4 + j0[2]);
            tb2 = cplx{w2.x, w2.y};
        }
    }
    if (A.ok0) {
        const double *src = p.in + A.in_base;
        const double *src1 = A.ok1 ? src + N : src;           // x: second line of the pair (a copy of the first if it does not exist)
#pragma unroll
        for (int it = 0; it < IT0; ++it)
#pragma unroll
            for (int r = 0; r < R0; ++r) {
                const int slot = slot_for(j0[it] + r * PER0);
                if (YP) {
                    const double2 w = *reinterpret_cast<const double2 *>(src + (size_t)slot * A.in_stride);
                    v[it * R0 + r] = cplx{w.x, w.y};
                } else {
                    v[it * R0 + r] = cplx{src[slot], src1[slot]};
                }
            }
    } else {
#pragma unroll
        for (int q = 0; q < 16; ++q) v[q] = cplx{0.0, 0.0};
    }
#pragma unroll
    for (int it = 0; it < IT0; ++it)
#pragma unroll
        for (int r = 0; r < R0; ++r) {
            const double sc = special_slot<BC, N>(slot_for(j0[it] + r * PER0)) ? p.s0 : p.s1;
            v[it * R0 + r] = cplx{sc * v[it * R0 + r].x, sc * v[it * R0 + r].y};
        }
    // (zk, zm) hold the coefficients of bins k and N - k on entry, Z_k and Z_{N-k} on exit;  0 < k < N, k != N/2
    auto build = [&](int k, cplx tk, cplx &zk, cplx &zm) {
        if (BC == 2) {
            const cplx ar = k < N / 2 ? zk : zm, ai = k < N / 2 ? zm : zk;   // B_kk = (ar - i ai) / 2, B_{N-kk} = (ar + i ai) / 2 per line
            const cplx lo{0.5 * (ar.x + ai.y), 0.5 * (ar.y - ai.x)}, hi{0.5 * (ar.x - ai.y), 0.5 * (ar.y + ai.x)};
            zk = k < N / 2 ? lo : hi;
            zm = k < N / 2 ? hi : lo;
        } else {
            const cplx ak = zk, am = zm;
            const cplx tm{-tk.y, -tk.x};                         // e^{-i pi (N-k) / 2N} = -i conj tk
            // B_k = e^{+i pi k / 2N} (a_k - i a_{N-k}) / 2 per line; Z = B_1 + i B_2
            const cplx b1 = cmul(cplx{0.5 * tk.x, -0.5 * tk.y}, cplx{ak.x, -am.x}), b2 = cmul(cplx{0.5 * tk.x, -0.5 * tk.y}, cplx{ak.y, -am.y});
            zk = cplx{b1.x - b2.y, b1.y + b2.x};
            const cplx c1 = cmul(cplx{0.5 * tm.x, -0.5 * tm.y}, cplx{am.x, -ak.x}), c2 = cmul(cplx{0.5 * tm.x, -0.5 * tm.y}, cplx{am.y, -ak.y});
            zm = cplx{c1.x - c2.y, c1.y + c2.x};
        }
    };
    if (R0 == 4) {
#pragma unroll
        for (int r = 0; r < R0; ++r) build(j0[2] + r * PER0, cmul(tb2, rot<R0>(r)), v[2 * R0 + r], v[3 * R0 + R0 - 1 - r]);
    }
    if (u) {
#pragma unroll
        for (int r = 0; r < R0; ++r) build(j0[0] + r * PER0, cmul(tb0, rot<R0>(r)), v[r], v[R0 + R0 - 1 - r]);
    } else {
        // bins 0 and N/2 are their own partners: B_0 = a_0 and (cosine / sine) B_{N/2} = e^{+i pi / 4} (a - i a) / 2 = a / sqrt 2
        if (BC != 2) v[R0 / 2] = cplx{0.70710678118654752440 * v[R0 / 2].x, 0.70710678118654752440 * v[R0 / 2].y};
#pragma unroll
        for (int r = 1; r < R0 / 2; ++r) build(r * PER0, rot<R0>(r), v[r], v[R0 - r]);
#pragma unroll
        for (int r = 0; r < R0 / 2; ++r) build(PER0 / 2 + r * PER0, cmul(rot_half<R0>(), rot<R0>(r)), v[R0 + r], v[R0 + R0 - 1 - r]);
    }
#pragma unroll
    for (int it = 0; it < IT0; ++it) {
        bfly<R0, 1>(v + it * R0);
#pragma unroll
        for (int r = 0; r < R0; ++r) seq[padf<LOGN, 1>(j0[it] * R0 + r)] = v[it * R0 + r];
    }
    __syncthreads();
    middle_passes<LOGN, 1, 1, R0, UPP, !YP>(seq, v, p, u);

    // ---- last pass ------------------------------------------------------------------------------------------------------
    constexpr int RL = radix_at(LOGN, NP - 1, 1), ITL = 16 / RL, NSL = N / RL;
#pragma unroll
    for (int it = 0; it < ITL; ++it) {
        const int j = u + it * UPP;
#pragma unroll
        for (int r = 0; r < RL; ++r) v[it * RL + r] = seq[padf<LOGN, 1>(j + r * NSL)];
        twiddle<RL, 1, (!YP && NSL >= 32)>(v + it * RL, p.Wq[NP - 1], NSL, j);
        bfly<RL, 1>(v + it * RL);
    }
    if (YP) {       // z[n] -> sample i(n) of both lines: one 16-byte store per row
#pragma unroll
        for (int it = 0; it < ITL; ++it)
#pragma unroll
            for (int r = 0; r < RL; ++r) {
                double sg;
                const int i = sample_of<BC, N>(u + it * UPP + r * NSL, sg);
                if (A.ok0) *reinterpret_cast<double2 *>(p.out + A.out_base + (size_t)i * A.out_stride) = make_double2(sg * v[it * RL + r].x, sg * v[it * RL + r].y);
            }
    } else if (BC == 2) {
        // x, periodic: z[n] is sample n — 8-byte stores contiguous across the lanes, straight from the registers (0.355 -> 0.315 ms
        // at 512^3; for the cosine / sine orders the same stores would be stride-2 and lose to the staged rows: 0.400 vs 0.344 ms)
#pragma unroll
        for (int it = 0; it < ITL; ++it)
#pragma unroll
            for (int r = 0; r < RL; ++r) {
                double sg;
                const int i = sample_of<BC, N>(u + it * UPP + r * NSL, sg);
                if (A.ok0) p.out[A.out_base + i] = sg * v[it * RL + r].x;
                if (A.ok1) p.out[A.out_base + N + i] = sg * v[it * RL + r].y;
            }
    } else {
        __syncthreads();
#pragma unroll
        for (int it = 0; it < ITL; ++it)
#pragma unroll
            for (int r = 0; r < RL; ++r) seq[padf<LOGN, 1>(u + it * UPP + r * NSL)] = v[it * RL + r];
        __syncthreads();
        constexpr int STEPS = G::PAIRS * (N / 2);
#pragma unroll 4
        for (int e = t; e < STEPS; e += G::THREADS) {
            const int q = e >> (LOGN - 1), i = (e & (N / 2 - 1)) << 1;
            const int l = blockIdx.x * G::LINES + 2 * q;
            const cplx *z = buf + q * NPAD;
            cplx c0, c1;
            double s1 = 1.0;
            if (BC == 2) {
                c0 = z[padf<LOGN, 1>(i)];
                c1 = z[padf<LOGN, 1>(i + 1)];
            } else {
                c0 = z[padf<LOGN, 1>(i >> 1)];
                c1 = z[padf<LOGN, 1>(N - 1 - (i >> 1))];
                if (BC == 1) s1 = -1.0;
            }
            if (l < p.lines) *reinterpret_cast<double2 *>(p.out + ((size_t)l << LOGN) + i) = make_double2(c0.x, s1 * c1.x);
            if (l + 1 < p.lines) *reinterpret_cast<double2 *>(p.out + ((size_t)(l + 1) << LOGN) + i) = make_double2(c0.y, s1 * c1.y);
        }
    }
}

}  // namespace

// pass radices of a length-2^m transform (radix_at above), forward or inverse order
static int fft_radices(int n, int radix[4], int inv) {
    int m = 0;
    while ((1 << m) < n) ++m;
    for (int q = 0; q < 4; ++q) radix[q] = radix_at(m, q, inv);
    return m;
}

bool fft_supported(int n) { return n >= 16 && n <= 2048 && (n & (n - 1)) == 0; }

// Host side of the twiddle tables, interleaved (re, im): T4[k] = e^{-i pi k / 2N} (n entries), then for every pass
// after the first its table e^{-2 pi i r k / (Ns R)}, r = 1..R-1, k = 0..Ns-1 — for the forward radix order, then (where
// it differs: n >= 1024) for the inverse order.
static void pass_tables(int n, int inv, std::vector<double> &out) {
    const long double pi = 3.14159265358979323846264338327950288L;
    int radix[4];
    fft_radices(n, radix, inv);
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
static bool orders_differ(int n) {
    int f[4], i[4];
    fft_radices(n, f, 0);
    fft_radices(n, i, 1);
    for (int q = 0; q < 4; ++q)
        if (f[q] != i[q]) return true;
    return false;
}
void fft_tables(int n, std::vector<double> &out) {
    const long double pi = 3.14159265358979323846264338327950288L;
    out.clear();
    for (int t = 0; t < n; ++t) {
        const long double b = -pi * t / (2.0L * n);
        out.push_back((double)cosl(b));
        out.push_back((double)sinl(b));
    }
    pass_tables(n, 0, out);
    if (orders_differ(n)) pass_tables(n, 1, out);
}

cudaError_t fft_configure() { return cudaSuccess; }   // shared-memory opt-in happens per instantiation at first launch

namespace {

template <bool YP, int LOGN, int BC>
cudaError_t launch_bc(const FftParams &p, int inverse, cudaStream_t stream) {
    using G = Geo<YP, LOGN>;
    constexpr int threads = G::THREADS;
    constexpr size_t smem = G::SMEM;
    int grid_x, grid_y = 1;
    if (YP) {
        const int ncols = p.bgroups * 16;      // columns of this launch (set by launch_fft, a multiple of COLS)
        if (ncols % G::COLS) return cudaErrorInvalidValue;
        grid_x = ncols / G::COLS;
        grid_y = (p.planes + G::PL - 1) / G::PL;
    } else {
        grid_x = (p.lines + G::LINES - 1) / G::LINES;
    }
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
    if (inverse) return launch_pdl(fft_inverse_kernel<YP, LOGN, BC>, grid, dim3(threads), smem, stream, p);
    if (YP && p.npeers) {
        if (smem > 48 * 1024) {
            static DeviceOnce configured_peers;
            cudaError_t e = configured_peers.run([&] {
                return cudaFuncSetAttribute(fft_forward_kernel<YP, LOGN, BC, YP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            });
            if (e != cudaSuccess) return e;
        }
        return launch_pdl(fft_forward_kernel<YP, LOGN, BC, YP>, grid, dim3(threads), smem, stream, p);
    }
    return launch_pdl(fft_forward_kernel<YP, LOGN, BC>, grid, dim3(threads), smem, stream, p);
}

template <bool YP, int LOGN>
cudaError_t launch_one(const FftParams &p, int inverse, cudaStream_t stream) {
    if (p.bc == 0) return launch_bc<YP, LOGN, 0>(p, inverse, stream);
    if (p.bc == 1) return launch_bc<YP, LOGN, 1>(p, inverse, stream);
    return launch_bc<YP, LOGN, 2>(p, inverse, stream);
}

template <bool YP>
cudaError_t launch_len(const FftParams &p, int inverse, cudaStream_t stream) {
    switch (p.logN) {
        case 4: return launch_one<YP, 4>(p, inverse, stream);
        case 5: return launch_one<YP, 5>(p, inverse, stream);
        case 6: return launch_one<YP, 6>(p, inverse, stream);
        case 7: return launch_one<YP, 7>(p, inverse, stream);
        case 8: return launch_one<YP, 8>(p, inverse, stream);
        case 9: return launch_one<YP, 9>(p, inverse, stream);
        case 10: return launch_one<YP, 10>(p, inverse, stream);
        case 11: return launch_one<YP, 11>(p, inverse, stream);
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
    if (a.npeers) {
        if (a.npeers < 0 || a.npeers > MAX_PEERS || !p.blk_out || a.ny % 16) return cudaErrorInvalidValue;
        p.npeers = a.npeers;
        p.units = a.ny / 16;
        for (int q = 0; q < a.npeers; ++q) {
            if (!a.peer_out[q]) return cudaErrorInvalidValue;
            p.peer_out[q] = a.peer_out[q];
        }
    }
    p.nz = a.nz; p.k0 = a.k0;
    {
        const double2 *w = p.T4 + N;
        // forward-order tables first; the inverse-order set follows where the orders differ
        for (int dir = 0; dir <= (a.inverse && orders_differ(N) ? 1 : 0); ++dir) {
            p.logN = fft_radices(N, p.radix, dir);
            int Ns = 1;
            for (int q = 0; q < 4 && p.radix[q]; ++q) {
                p.Wq[q] = w;
                if (q > 0) w += (p.radix[q] - 1) * Ns;
                Ns *= p.radix[q];
            }
        }
    }
    p.planes = a.planes;
    if (a.dir == 0) {
        p.lines = a.ny * a.planes;
        return launch_len<false>(p, a.inverse, stream);
    }
    const int ncols = a.ncols ? a.ncols : a.nx;
    if (ncols % 16 || a.x0 % 16 || a.x0 < 0 || a.x0 + ncols > a.nx) return cudaErrorInvalidValue;
    p.bgroups = ncols / 16;
    // the natural-layout side starts at column x0 of every row; the blocked side is indexed by the slab-local column
    if (!p.blk_in) p.in += a.x0;
    if (!p.blk_out) p.out += a.x0;
    return launch_len<true>(p, a.inverse, stream);
}

}  // namespace tpt
