// projection.cu — the staggered-grid operators around the pressure solve of the fractional-step method,
// Eq. 2c–2e (staggered arrangement PAPER.md:57):
//   divergence_kernel   rhs = scale * D(u, v, w)                 right-hand side of Eq. 2c (scale = 1/(gamma_k dt))
//   correct_kernel      u -= c G Phi  (Eq. 2d)  and, fused,  P += Phi - alpha L_I Phi  (Eq. 2e)
// Layout (reading A18): u (nz, ny, nx+1) on x-faces, v (nz, ny+1, nx) on y-faces, w (nz+1, ny, nx) on
// z-faces; face f lies between cells f-1 and f.  Boundary faces: Neumann = wall (gradient 0, the face keeps its
// prescribed value), Dirichlet = ghost value -Phi at one cell width, periodic = faces 0 and n are one face (entry n
// ignored on input, written as a copy of entry 0).
//
// Both kernels are HBM-bound stencils: one thread per two x-neighbouring cells of one z-level (16-byte accesses; the
// one-cell-per-thread kernels serve odd nx), x contiguous across the warp, the x / y / z
// neighbours re-read through L1/L2.  Algorithmic traffic: divergence 32 B/pt (three face arrays in, one cell array
// out), correction 56 B/pt (Phi in, three face arrays read-modify-write) + 16 B/pt with the pressure update.
#include "kernels.cuh"

namespace tpt {

namespace {

constexpr int PX = 128;   // threads per block, along x
constexpr int KZD = 16;   // z-levels per thread (divergence)

__global__ void __launch_bounds__(PX, 8)
divergence_kernel(const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                  const double *__restrict__ rwx, const double *__restrict__ rwy, const double *__restrict__ rwz,
                  double *__restrict__ out, int nx, int ny, int nz, int px, int py, int pz, double scale) {
    const int i = blockIdx.x * PX + threadIdx.x;
    const int j = blockIdx.y;
    const int k0 = blockIdx.z * KZD;
    if (i >= nx) return;
    const int k1 = min(k0 + KZD, nz);
    const size_t plane = (size_t)nx * ny;
    const int ih = (px && i == nx - 1) ? 0 : i + 1;   // periodic: face n is face 0
    const int jh = (py && j == ny - 1) ? 0 : j + 1;
    const double rx = rwx[i], ry = rwy[j];
    double wlo = w[i + (size_t)nx * j + plane * k0];
#pragma unroll 4
    for (int k = k0; k < k1; ++k) {
        const size_t urow = (size_t)(nx + 1) * (j + (size_t)ny * k);
        const size_t vpl = (size_t)nx * (ny + 1) * k;
        const double whi = w[i + (size_t)nx * j + plane * ((pz && k == nz - 1) ? 0 : k + 1)];   // periodic: face nz is face 0
        const double du = (u[urow + ih] - u[urow + i]) * rx;
        const double dv = (v[vpl + (size_t)nx * jh + i] - v[vpl + (size_t)nx * j + i]) * ry;
        const double dw = (whi - wlo) * rwz[k];
        out[i + (size_t)nx * j + plane * k] = scale * (du + dv + dw);
        wlo = whi;
    }
}

// Even nx: two cells per thread, 16-byte accesses on v, w and out (the u rows have odd length: 8-byte accesses).
__global__ void __launch_bounds__(PX)
divergence2_kernel(const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                   const double *__restrict__ rwx, const double *__restrict__ rwy, const double *__restrict__ rwz,
                   double *__restrict__ out, int nx, int ny, int nz, int px, int py, int pz, double scale) {
    const int i = 2 * (blockIdx.x * PX + threadIdx.x);
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= nx) return;
    const size_t plane = (size_t)nx * ny;
    const size_t wo = i + (size_t)nx * j + plane * k;
    const size_t urow = (size_t)(nx + 1) * (j + (size_t)ny * k);
    const size_t vo = (size_t)nx * (ny + 1) * k + (size_t)nx * j + i;
    const int jh = (py && j == ny - 1) ? -j : 1;                  // periodic: face ny is face 0
    const double u0 = u[urow + i], u1 = u[urow + i + 1];
    const double u2 = u[urow + ((px && i == nx - 2) ? 0 : i + 2)];
    const double2 vl = *reinterpret_cast<const double2 *>(v + vo);
    const double2 vh = *reinterpret_cast<const double2 *>(v + vo + (ptrdiff_t)nx * jh);
    const double2 wl = *reinterpret_cast<const double2 *>(w + wo);
    const double2 wh = *reinterpret_cast<const double2 *>((pz && k == nz - 1) ? w + wo - plane * k : w + wo + plane);
    const double ry = rwy[j], rz = rwz[k];
    double2 o;
    o.x = scale * ((u1 - u0) * rwx[i] + (vh.x - vl.x) * ry + (wh.x - wl.x) * rz);
    o.y = scale * ((u2 - u1) * rwx[i + 1] + (vh.y - vl.y) * ry + (wh.y - wl.y) * rz);
    *reinterpret_cast<double2 *>(out + wo) = o;
}

// ghost value beyond a non-periodic boundary (mirror ghost cell, A3): Neumann +phi, Dirichlet -phi
__device__ __forceinline__ double ghost(int bc, double phi) { return bc == 1 ? -phi : phi; }

// gf* = 1 / centre spacing at every face (boundary faces: one cell width; periodic: the wrap spacing, A17).
template <bool WITH_P, int KZ>
__global__ void __launch_bounds__(PX)
correct_kernel(const double *__restrict__ phi, double *__restrict__ u, double *__restrict__ v, double *__restrict__ w,
               double *__restrict__ p, const double *__restrict__ gfx, const double *__restrict__ gfy,
               const double *__restrict__ gfz, const double *__restrict__ rwx, const double *__restrict__ rwy,
               const double *__restrict__ rwz, int nx, int ny, int nz, int bcx, int bcy, int bcz, double c,
               double alpha, int dirs) {
    const int i = blockIdx.x * PX + threadIdx.x;
    const int j = blockIdx.y;
    const int k0 = blockIdx.z * KZ;
    if (i >= nx) return;
    const int k1 = min(k0 + KZ, nz);
    const size_t plane = (size_t)nx * ny;
    const bool px = bcx == 2, py = bcy == 2, pz = bcz == 2;
    const double gxl = gfx[i], gxh = gfx[i + 1], gyl = gfy[j], gyh = gfy[j + 1];
    const size_t col = i + (size_t)nx * j;
    double cur = phi[col + plane * k0];
    double below = k0 > 0 ? phi[col + plane * (k0 - 1)] : (pz ? phi[col + plane * (nz - 1)] : ghost(bcz, cur));
    for (int k = k0; k < k1; ++k) {
        const double *row = phi + (size_t)nx * j + plane * k;     // this x-line
        const double *pl = phi + plane * k + i;                   // this (i, :) line of the plane
        const double xm = i > 0 ? row[i - 1] : (px ? row[nx - 1] : ghost(bcx, cur));
        const double ym = j > 0 ? pl[(size_t)nx * (j - 1)] : (py ? pl[(size_t)nx * (ny - 1)] : ghost(bcy, cur));
        const double above = k < nz - 1 ? phi[col + plane * (k + 1)] : (pz ? phi[col] : ghost(bcz, cur));
        const double Gxl = gxl * (cur - xm), Gyl = gyl * (cur - ym), Gzl = gfz[k] * (cur - below);
        // Eq. 2d on the low faces of this cell
        const size_t uo = (size_t)(nx + 1) * (j + (size_t)ny * k) + i;
        const size_t vo = (size_t)nx * (ny + 1) * k + (size_t)nx * j + i;
        const size_t wo = col + plane * k;
        const double un = fma(-c, Gxl, u[uo]);
        u[uo] = un;
        const double vn = fma(-c, Gyl, v[vo]);
        v[vo] = vn;
        const double wn = fma(-c, Gzl, w[wo]);
        w[wo] = wn;
        if (pz && k == 0) w[wo + plane * nz] = wn;
        if (px && i == 0) u[uo + nx] = un;                        // periodic: face n is a copy of face 0
        if (py && j == 0) v[vo + (size_t)nx * ny] = vn;
        const bool xe = i == nx - 1, ye = j == ny - 1, ze = k == nz - 1;
        if (WITH_P || (xe && bcx == 1) || (ye && bcy == 1) || (ze && bcz == 1)) {
            const double xp = !xe ? row[i + 1] : (px ? row[0] : ghost(bcx, cur));
            const double yp = !ye ? pl[(size_t)nx * (j + 1)] : (py ? pl[0] : ghost(bcy, cur));
            const double Gxh = gxh * (xp - cur), Gyh = gyh * (yp - cur), Gzh = gfz[k + 1] * (above - cur);
            // high boundary faces (Dirichlet: corrected; Neumann: a wall, untouched; periodic: written above)
            if (xe && bcx == 1) u[uo + 1] = fma(-c, Gxh, u[uo + 1]);
            if (ye && bcy == 1) v[vo + nx] = fma(-c, Gyh, v[vo + nx]);
            if (ze && bcz == 1) w[wo + plane] = fma(-c, Gzh, w[wo + plane]);
            if (WITH_P) {                                         // Eq. 2e: P += Phi - alpha L_I Phi, L_I in flux form
                double lap = (Gzh - Gzl) * rwz[k];
                if (dirs & 1) lap += (Gxh - Gxl) * rwx[i];
                if (dirs & 2) lap += (Gyh - Gyl) * rwy[j];
                p[wo] += fma(-alpha, lap, cur);
            }
        }
        below = cur;
        cur = above;
    }
}

// The same for even nx with two x-neighbouring cells per thread: Phi, v, w and p move as 16-byte accesses (their rows
// are 16-byte aligned); the u rows have odd length nx + 1, so the two u faces are 8-byte accesses.  One z-level per
// thread (the z neighbours come from L2, which holds many planes).
template <bool WITH_P>
__global__ void __launch_bounds__(PX, 12)
correct2_kernel(const double *__restrict__ phi, double *__restrict__ u, double *__restrict__ v, double *__restrict__ w,
                double *__restrict__ p, const double *__restrict__ gfx, const double *__restrict__ gfy,
                const double *__restrict__ gfz, const double *__restrict__ rwx, const double *__restrict__ rwy,
                const double *__restrict__ rwz, int nx, int ny, int nz, int bcx, int bcy, int bcz, double c,
                double alpha, int dirs) {
    const int i = 2 * (blockIdx.x * PX + threadIdx.x);
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= nx) return;
    const size_t plane = (size_t)nx * ny;
    const bool px = bcx == 2, py = bcy == 2, pz = bcz == 2;
    const size_t wo = i + (size_t)nx * j + plane * k;
    const double *row = phi + (size_t)nx * j + plane * k;
    const double2 cur = *reinterpret_cast<const double2 *>(phi + wo);
    const double xm = i > 0 ? row[i - 1] : (px ? row[nx - 1] : ghost(bcx, cur.x));
    double2 ym, below;
    if (j > 0) ym = *reinterpret_cast<const double2 *>(phi + wo - nx);
    else if (py) ym = *reinterpret_cast<const double2 *>(phi + wo + (size_t)nx * (ny - 1));
    else ym = make_double2(ghost(bcy, cur.x), ghost(bcy, cur.y));
    if (k > 0) below = *reinterpret_cast<const double2 *>(phi + wo - plane);
    else if (pz) below = *reinterpret_cast<const double2 *>(phi + wo + plane * (nz - 1));
    else below = make_double2(ghost(bcz, cur.x), ghost(bcz, cur.y));
    const double g0 = gfx[i], g1 = gfx[i + 1], gyl = gfy[j], gzl = gfz[k];
    const double Gx0 = g0 * (cur.x - xm), Gx1 = g1 * (cur.y - cur.x);
    const double Gy0 = gyl * (cur.x - ym.x), Gy1 = gyl * (cur.y - ym.y);
    const double Gz0 = gzl * (cur.x - below.x), Gz1 = gzl * (cur.y - below.y);
    const size_t uo = (size_t)(nx + 1) * (j + (size_t)ny * k) + i;
    const size_t vo = (size_t)nx * (ny + 1) * k + (size_t)nx * j + i;
    const double un0 = fma(-c, Gx0, u[uo]), un1 = fma(-c, Gx1, u[uo + 1]);
    u[uo] = un0;
    u[uo + 1] = un1;
    double2 vv = *reinterpret_cast<double2 *>(v + vo);
    vv.x = fma(-c, Gy0, vv.x);
    vv.y = fma(-c, Gy1, vv.y);
    *reinterpret_cast<double2 *>(v + vo) = vv;
    double2 ww = *reinterpret_cast<double2 *>(w + wo);
    ww.x = fma(-c, Gz0, ww.x);
    ww.y = fma(-c, Gz1, ww.y);
    *reinterpret_cast<double2 *>(w + wo) = ww;
    if (pz && k == 0) *reinterpret_cast<double2 *>(w + wo + plane * nz) = ww;
    if (px && i == 0) u[uo + nx] = un0;
    if (py && j == 0) *reinterpret_cast<double2 *>(v + vo + (size_t)nx * ny) = vv;
    const bool xe = i == nx - 2, ye = j == ny - 1, ze = k == nz - 1;
    if (WITH_P || (xe && bcx == 1) || (ye && bcy == 1) || (ze && bcz == 1)) {
        const double xp = !xe ? row[i + 2] : (px ? row[0] : ghost(bcx, cur.y));
        double2 yp, above;
        if (!ye) yp = *reinterpret_cast<const double2 *>(phi + wo + nx);
        else if (py) yp = *reinterpret_cast<const double2 *>(phi + wo - (size_t)nx * (ny - 1));
        else yp = make_double2(ghost(bcy, cur.x), ghost(bcy, cur.y));
        if (!ze) above = *reinterpret_cast<const double2 *>(phi + wo + plane);
        else if (pz) above = *reinterpret_cast<const double2 *>(phi + wo - plane * k);
        else above = make_double2(ghost(bcz, cur.x), ghost(bcz, cur.y));
        const double gyh = gfy[j + 1], gzh = gfz[k + 1];
        const double Gx2 = gfx[i + 2] * (xp - cur.y);
        const double Gyh0 = gyh * (yp.x - cur.x), Gyh1 = gyh * (yp.y - cur.y);
        const double Gzh0 = gzh * (above.x - cur.x), Gzh1 = gzh * (above.y - cur.y);
        if (xe && bcx == 1) u[uo + 2] = fma(-c, Gx2, u[uo + 2]);
        if (ye && bcy == 1) {
            double2 t = *reinterpret_cast<double2 *>(v + vo + nx);
            t.x = fma(-c, Gyh0, t.x);
            t.y = fma(-c, Gyh1, t.y);
            *reinterpret_cast<double2 *>(v + vo + nx) = t;
        }
        if (ze && bcz == 1) {
            double2 t = *reinterpret_cast<double2 *>(w + wo + plane);
            t.x = fma(-c, Gzh0, t.x);
            t.y = fma(-c, Gzh1, t.y);
            *reinterpret_cast<double2 *>(w + wo + plane) = t;
        }
        if (WITH_P) {
            const double rz = rwz[k];
            double l0 = (Gzh0 - Gz0) * rz, l1 = (Gzh1 - Gz1) * rz;
            if (dirs & 1) { l0 += (Gx1 - Gx0) * rwx[i]; l1 += (Gx2 - Gx1) * rwx[i + 1]; }
            if (dirs & 2) { const double ry = rwy[j]; l0 += (Gyh0 - Gy0) * ry; l1 += (Gyh1 - Gy1) * ry; }
            double2 pp = *reinterpret_cast<double2 *>(p + wo);
            pp.x += fma(-alpha, l0, cur.x);
            pp.y += fma(-alpha, l1, cur.y);
            *reinterpret_cast<double2 *>(p + wo) = pp;
        }
    }
}

}  // namespace

// The two-cells-per-thread kernels make 16-byte accesses to every array but u (whose rows have odd length nx + 1);
// a pointer that is only 8-byte aligned (a view into a larger buffer) takes the one-cell kernels instead of faulting.
static bool aligned16(const void *q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; }

cudaError_t launch_divergence(const double *u, const double *v, const double *w, const ProjGeom &g, double scale,
                              double *out, cudaStream_t stream) {
    if (g.nx % 2 == 0 && aligned16(v) && aligned16(w) && aligned16(out)) {
        dim3 grid2((g.nx / 2 + PX - 1) / PX, g.ny, g.nz);
        divergence2_kernel<<<grid2, PX, 0, stream>>>(u, v, w, g.rwx, g.rwy, g.rwz, out, g.nx, g.ny, g.nz, g.bc[0] == 2,
                                                     g.bc[1] == 2, g.bc[2] == 2, scale);
        return cudaGetLastError();
    }
    dim3 grid((g.nx + PX - 1) / PX, g.ny, (g.nz + KZD - 1) / KZD);
    divergence_kernel<<<grid, PX, 0, stream>>>(u, v, w, g.rwx, g.rwy, g.rwz, out, g.nx, g.ny, g.nz, g.bc[0] == 2,
                                               g.bc[1] == 2, g.bc[2] == 2, scale);
    return cudaGetLastError();
}

cudaError_t launch_correct(const double *phi, double *u, double *v, double *w, double *p, const ProjGeom &g, double c,
                           double alpha, int dirs, cudaStream_t stream) {
    if (g.nx % 2 == 0 && aligned16(phi) && aligned16(v) && aligned16(w) && aligned16(p)) {   // two cells per thread, 16-byte accesses
        dim3 grid((g.nx / 2 + PX - 1) / PX, g.ny, g.nz);
        if (p)
            correct2_kernel<true><<<grid, PX, 0, stream>>>(phi, u, v, w, p, g.gfx, g.gfy, g.gfz, g.rwx, g.rwy, g.rwz, g.nx, g.ny,
                                                           g.nz, g.bc[0], g.bc[1], g.bc[2], c, alpha, dirs);
        else
            correct2_kernel<false><<<grid, PX, 0, stream>>>(phi, u, v, w, nullptr, g.gfx, g.gfy, g.gfz, g.rwx, g.rwy, g.rwz,
                                                            g.nx, g.ny, g.nz, g.bc[0], g.bc[1], g.bc[2], c, alpha, dirs);
    } else {
        dim3 grid((g.nx + PX - 1) / PX, g.ny, g.nz);
        if (p)
            correct_kernel<true, 1><<<grid, PX, 0, stream>>>(phi, u, v, w, p, g.gfx, g.gfy, g.gfz, g.rwx, g.rwy, g.rwz, g.nx,
                                                             g.ny, g.nz, g.bc[0], g.bc[1], g.bc[2], c, alpha, dirs);
        else
            correct_kernel<false, 1><<<grid, PX, 0, stream>>>(phi, u, v, w, nullptr, g.gfx, g.gfy, g.gfz, g.rwx, g.rwy, g.rwz,
                                                              g.nx, g.ny, g.nz, g.bc[0], g.bc[1], g.bc[2], c, alpha, dirs);
    }
    return cudaGetLastError();
}

}  // namespace tpt
