// star_sums.cuh — the star sums of Eq. 15 / Eq. 19 as device code shared by the
// Aberth kernels (aberth.cu) and the far-field module (fmm.cu):
//   S1 = sum_i 1/(z-z_i),  S2 = sum_i m_i/(z-z_i)^2,  S3 = sum_i m_i/(z-z_i)^3,  Sm = sum_i m_i/(z-z_i),
// either directly (pair_star, one star at a time) or split as in PAPER.md:188-195 (§4.1) into the stars
// near the point, summed directly, and the distant ones, read off a Taylor series of the point's grid
// node (fmm_star_sums).  Product path only; the oracle has its own straight loops.
#pragma once
#include "mlcc_common.cuh"

namespace mlcc {

struct StarAcc {
    double s1x, s1y;   // S1
    double s2x, s2h;   // Re S2, (Im S2)/2
    double s3x, s3y;   // S3
    double smx, smy;   // Sm = sum m/(z-z_i) (its conjugate is the deflection of Eq. 12; only with CAUS)
};

// Uniform grid of nodes over the stars' bounding square and, for every node, the Taylor series about
// its centre c of the sums over the stars that are NOT in the (2h+1)^2 nodes around it:
//   sum_far m_i/(z - z_i) = (1/s) sum_l Lm[l] u^l,   u = (z - c)/s,   Lm[l] = -sum_far m_i (s/(z_i - c))^(l+1),
// and L1 the same with m_i = 1.  Lengths are scaled by the node size s so that |u| <= 1/sqrt(2) and
// |s/(z_i - c)| <= 1/(h + 1/2): the terms fall like rho^l, rho = (1/sqrt 2)/(h + 1/2) (0.283 for h = 2).
struct FmmGeom {      // written on the device by the build
    double x0, y0;    // lower-left corner of the grid
    double s, inv_s;  // node size and its reciprocal
};
struct FmmGrid {
    const FmmGeom *geom;      // [1]
    int G;                    // nodes per side
    int P1;                   // Taylor coefficients per node (order P1 - 1), a multiple of 8
    int h;                    // half-width of the near neighbourhood in nodes
    int N;                    // stars
    const int *cell_start;    // [G*G + 1] first sorted star of every node (row-major, y outer)
    const double2 *sxy;       // [N] stars sorted by node, original order inside a node
    const double *sm;         // [N]
    const double2 *Lm;        // [G*G][P1]
    const double2 *L1;        // [G*G][P1]
};

#ifdef __CUDACC__

// (root, star): with d = z - z_i, w = 1/d = conj(d)/|d|^2 = (wx, wy)  [dy is taken as y_i - y],
//   S1 += w,  S2 += m w^2 = m (wx^2 - wy^2, 2 wx wy),  S3 += m w^3 = m (wx (wx^2 - 3 wy^2), wy (3 wx^2 - wy^2)).
// 22 FP64 instructions + 1 MUFU; 18 of them name at most two distinct register sources.
// WITH_S1 = false leaves S1 out (the iterations without the Aberth sum take the Newton step of F, which needs
// neither A nor S1: DESIGN.md R27): 20 (22) FP64 instructions.
template <bool CAUS, bool WITH_S1 = true>
__device__ __forceinline__ void pair_star(double zx, double zy, double2 s, double m, StarAcc &a)
{
    const double dx = zx - s.x;
    const double dy = s.y - zy;
    const double r2 = fma(dy, dy, dx * dx);
    const double inv = rcp_full(r2);
    const double wx = dx * inv;
    const double wy = dy * inv;
    if (WITH_S1) {
        a.s1x += wx;
        a.s1y += wy;
    }
    const double ux = m * wx;
    const double uy = m * wy;
    if (CAUS) {
        a.smx += ux;
        a.smy += uy;
    }
    const double A = wx * wx;
    const double B = wy * wy;
    const double g = fma(-3.0, B, A);
    const double h = fma(3.0, A, -B);
    const double c = A - B;
    a.s2x = fma(m, c, a.s2x);
    a.s2h = fma(ux, wy, a.s2h);
    a.s3x = fma(ux, g, a.s3x);
    a.s3y = fma(uy, h, a.s3y);
}

// The same for a field of EQUAL masses m_i = m0 (BASELINE.json configs 1, 2, 5): the sums are accumulated
// unweighted and scaled once at the end (star_sums_scale), 20 FP64 instructions per pair instead of 24:
//   S1 += w,  S2/m0 += w^2,  S3/m0 += w^3,  Sm/m0 = S1.
// Where S1 is not wanted (WITH_S1 = false) but the caustic point is, w is added into the Sm fields instead.
// With m0 = 1 the results are bit-identical to pair_star (every product by the mass is exact there).
template <bool CAUS, bool WITH_S1 = true>
__device__ __forceinline__ void pair_star_eq(double zx, double zy, double2 s, StarAcc &a)
{
    const double dx = zx - s.x;
    const double dy = s.y - zy;
    const double r2 = fma(dy, dy, dx * dx);
    const double inv = rcp_full(r2);
    const double wx = dx * inv;
    const double wy = dy * inv;
    if (WITH_S1) {
        a.s1x += wx;
        a.s1y += wy;
    } else if (CAUS) {
        a.smx += wx;
        a.smy += wy;
    }
    const double A = wx * wx;
    const double B = wy * wy;
    const double g = fma(-3.0, B, A);
    const double h = fma(3.0, A, -B);
    a.s2x += A - B;
    a.s2h = fma(wx, wy, a.s2h);
    a.s3x = fma(wx, g, a.s3x);
    a.s3y = fma(wy, h, a.s3y);
}
template <bool CAUS, bool WITH_S1 = true>
__device__ __forceinline__ void star_sums_scale(StarAcc &a, double m0)
{
    if (CAUS) {
        a.smx = m0 * (WITH_S1 ? a.s1x : a.smx);
        a.smy = m0 * (WITH_S1 ? a.s1y : a.smy);
    }
    a.s2x *= m0; a.s2h *= m0;
    a.s3x *= m0; a.s3y *= m0;
}

// P(u) = sum_l a[l] u^l with its first two derivatives by one Horner pass (synthetic division):
// returns P, P', P''/2.
__device__ __forceinline__ void horner3(const double2 *__restrict__ a, int n, double ux, double uy,
                                        double2 &p0, double2 &p1, double2 &p2)
{
    double b0x = 0, b0y = 0, b1x = 0, b1y = 0, b2x = 0, b2y = 0;
#pragma unroll 8
    for (int l = n - 1; l >= 0; --l) {
        const double2 c = __ldg(&a[l]);
        double tx = fma(b2x, ux, fma(-b2y, uy, b1x));   // b2 = b2 u + b1
        double ty = fma(b2x, uy, fma(b2y, ux, b1y));
        b2x = tx; b2y = ty;
        tx = fma(b1x, ux, fma(-b1y, uy, b0x));          // b1 = b1 u + b0
        ty = fma(b1x, uy, fma(b1y, ux, b0y));
        b1x = tx; b1y = ty;
        tx = fma(b0x, ux, fma(-b0y, uy, c.x));          // b0 = b0 u + a_l
        ty = fma(b0x, uy, fma(b0y, ux, c.y));
        b0x = tx; b0y = ty;
    }
    p0 = make_double2(b0x, b0y);
    p1 = make_double2(b1x, b1y);
    p2 = make_double2(b2x, b2y);
}
__device__ __forceinline__ double2 horner1(const double2 *__restrict__ a, int n, double ux, double uy)
{
    double bx = 0, by = 0;
#pragma unroll 8
    for (int l = n - 1; l >= 0; --l) {
        const double2 c = __ldg(&a[l]);
        const double tx = fma(bx, ux, fma(-by, uy, c.x));
        const double ty = fma(bx, uy, fma(by, ux, c.y));
        bx = tx; by = ty;
    }
    return make_double2(bx, by);
}

// All four star sums at z = (zx, zy), near stars directly and distant stars from the node's Taylor
// series ("used in the calculation of w, F(z), and F'(z)").  Adds into `a` (all eight
// fields) and returns true.  A point outside the grid (the outer pair of roots at |z| ~ 2R,
// PAPER.md:422 fn. 7) or a non-finite one has no node: returns false and leaves `a` alone -- the caller
// sums such a point directly over all stars (fmm_direct_all, or a whole CTA per point in aberth.cu).
__device__ __forceinline__ bool fmm_star_sums(const FmmGrid &g, double zx, double zy, StarAcc &a)
{
    const FmmGeom ge = *g.geom;
    const double fx = (zx - ge.x0) * ge.inv_s, fy = (zy - ge.y0) * ge.inv_s;
    const bool inside = fx >= 0.0 && fy >= 0.0 && fx < (double)g.G && fy < (double)g.G;   // false for NaN
    if (!inside) return false;
    const int ix = (int)fx, iy = (int)fy;
    const int xa = max(ix - g.h, 0), xb = min(ix + g.h, g.G - 1);
    // The near stars of one node row are one contiguous range of the sorted arrays.  Four stars are loaded
    // before any is used (a star past the range is replaced by a massless one far away), so a thread that
    // runs alone -- the last unfrozen roots of a row -- waits for memory once per four pairs, not per pair.
    for (int cy = max(iy - g.h, 0); cy <= min(iy + g.h, g.G - 1); ++cy) {
        const int i0 = __ldg(&g.cell_start[cy * g.G + xa]), i1 = __ldg(&g.cell_start[cy * g.G + xb + 1]);
        for (int i = i0; i < i1; i += 4) {
            double2 s[4];
            double m[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const bool in = i + u < i1;
                const int q = in ? i + u : i;
                s[u] = __ldg(&g.sxy[q]);
                m[u] = in ? __ldg(&g.sm[q]) : 0.0;
                if (!in) s[u] = make_double2(1e150, 1e150);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) pair_star<true>(zx, zy, s[u], m[u], a);
        }
    }
    const double ux = fx - ((double)ix + 0.5), uy = fy - ((double)iy + 0.5);   // (z - c)/s
    const size_t node = (size_t)(iy * g.G + ix) * g.P1;
    double2 p0, p1, p2;
    horner3(g.Lm + node, g.P1, ux, uy, p0, p1, p2);
    const double2 q0 = horner1(g.L1 + node, g.P1, ux, uy);
    const double i1s = ge.inv_s, i2s = i1s * i1s, i3s = i2s * i1s;
    a.smx += p0.x * i1s;            // Sm  += Phi_m
    a.smy += p0.y * i1s;
    a.s2x -= p1.x * i2s;            // S2  += -Phi_m'
    a.s2h -= 0.5 * p1.y * i2s;
    a.s3x += p2.x * i3s;            // S3  += Phi_m''/2
    a.s3y += p2.y * i3s;
    a.s1x += q0.x * i1s;            // S1  += Phi_1
    a.s1y += q0.y * i1s;
    return true;
}

__device__ __forceinline__ void fmm_direct_all(const FmmGrid &g, double zx, double zy, StarAcc &a)
{
    for (int i = 0; i < g.N; ++i) pair_star<true>(zx, zy, g.sxy[i], g.sm[i], a);
}

#endif  // __CUDACC__

// host side (fmm.cu): builds the grid and the node series in `ws` on `stream`; no host synchronisation
int fmm_build(const double2 *stars, const double *masses, int N, int order, int stars_per_node,
              Workspace &ws, FmmGrid *out, cudaStream_t stream);

}  // namespace mlcc
