// Per-site mathematics of the two theories, written against a tile accessor
// T(c, dy, dx) = component c of the (stage) field at offset (dx, dy) from the site.
// Formulas: DESIGN.md "Discrete energies" (readings R1-R3, R9); stencils PAPER.md:104-109.
#pragma once
#include "ss_common.cuh"

namespace ss {

// weights of the halo rule in the site-form energy: 1 if the neighbour is interior, 2 if it
// lies in the frozen halo (DESIGN R3).  Index: 0:+1, 1:-1, 2:+2, 3:-2.
struct EdgeW {
  int x[4], y[4];
  __device__ __forceinline__ EdgeW(int gx, int gy, int Nx, int Ny) {
    x[0] = (gx + 1 < Nx - HALO) ? 1 : 2;
    x[1] = (gx - 1 >= HALO) ? 1 : 2;
    x[2] = (gx + 2 < Nx - HALO) ? 1 : 2;
    x[3] = (gx - 2 >= HALO) ? 1 : 2;
    y[0] = (gy + 1 < Ny - HALO) ? 1 : 2;
    y[1] = (gy - 1 >= HALO) ? 1 : 2;
    y[2] = (gy + 2 < Ny - HALO) ? 1 : 2;
    y[3] = (gy - 2 >= HALO) ? 1 : 2;
  }
  __device__ __forceinline__ int wx(int s) const { return x[s]; }
  __device__ __forceinline__ int wy(int s) const { return y[s]; }
};

// all neighbours interior (sites at least 4 from every edge): the weights fold away
struct BulkW {
  __device__ __forceinline__ constexpr int wx(int) const { return 1; }
  __device__ __forceinline__ constexpr int wy(int) const { return 1; }
};

// eq. (1) numerators: 12h * D f = 8 (f+1 - f-1) - (f+2 - f-2)
template <typename real>
__device__ __forceinline__ real d1n(real fm2, real fm1, real fp1, real fp2) {
  return real(8) * (fp1 - fm1) - (fp2 - fm2);
}

template <typename real, typename Tile>
__device__ __forceinline__ real Dxn(const Tile& T, int c) {
  return d1n<real>(T(c, 0, -2), T(c, 0, -1), T(c, 0, 1), T(c, 0, 2));
}
template <typename real, typename Tile>
__device__ __forceinline__ real Dyn(const Tile& T, int c) {
  return d1n<real>(T(c, -2, 0), T(c, -1, 0), T(c, 1, 0), T(c, 2, 0));
}
// eq. (2) numerators: 12h^2 * Lx f, 12h^2 * Ly f
template <typename real, typename Tile>
__device__ __forceinline__ real Lxn(const Tile& T, int c) {
  return real(16) * (T(c, 0, 1) + T(c, 0, -1)) - (T(c, 0, 2) + T(c, 0, -2)) - real(30) * T(c, 0, 0);
}
template <typename real, typename Tile>
__device__ __forceinline__ real Lyn(const Tile& T, int c) {
  return real(16) * (T(c, 1, 0) + T(c, -1, 0)) - (T(c, 2, 0) + T(c, -2, 0)) - real(30) * T(c, 0, 0);
}
// (12h)^2 * DxDy f on the 4x4 box of corner neighbours; W(dy,dx) optional weights
template <typename real, typename Tile>
__device__ __forceinline__ real Dxyn(const Tile& T, int c) {
  real col[4];
  const int ks[4] = {-2, -1, 1, 2};
#pragma unroll
  for (int q = 0; q < 4; ++q)
    col[q] = d1n<real>(T(c, -2, ks[q]), T(c, -1, ks[q]), T(c, 1, ks[q]), T(c, 2, ks[q]));
  return d1n<real>(col[0], col[1], col[2], col[3]);
}

// ------------------------------------------------------------------ chiral magnet
template <typename real>
struct CM {
  static constexpr int C = 3;

  // a = -(G - (G.n) n),  G = -(Lx+Ly) n + 2 kappa (Dy n3, -Dx n3, Dx n2 - Dy n1) - (B + 2K n3) e3
  // with the stencil weights folded into five constants (kernel parameters, so they are
  // constant-bank operands): lap0/1/2 = 60, 16, 1 /(12h^2); dm1/2 = 2 kappa (8, 1)/(12h).
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel(const Tile& T, const P& p, real B, real a[3]) {
    const real n1 = T(0, 0, 0), n2 = T(1, 0, 0), n3 = T(2, 0, 0);
    real G[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {  // -(Lx + Ly) n_c
      const real s1 = (T(c, 0, 1) + T(c, 0, -1)) + (T(c, 1, 0) + T(c, -1, 0));
      const real s2 = (T(c, 0, 2) + T(c, 0, -2)) + (T(c, 2, 0) + T(c, -2, 0));
      G[c] = p.lap2 * s2 + (p.lap0 * T(c, 0, 0) - p.lap1 * s1);
    }
    G[0] += p.dm1 * (T(2, 1, 0) - T(2, -1, 0)) - p.dm2 * (T(2, 2, 0) - T(2, -2, 0));
    G[1] -= p.dm1 * (T(2, 0, 1) - T(2, 0, -1)) - p.dm2 * (T(2, 0, 2) - T(2, 0, -2));
    G[2] += p.dm1 * ((T(1, 0, 1) - T(1, 0, -1)) - (T(0, 1, 0) - T(0, -1, 0))) -
            p.dm2 * ((T(1, 0, 2) - T(1, 0, -2)) - (T(0, 2, 0) - T(0, -2, 0)));
    G[2] -= B + p.K2 * n3;
    const real gn = (G[0] * n1 + G[1] * n2) + G[2] * n3;
    a[0] = gn * n1 - G[0];
    a[1] = gn * n2 - G[1];
    a[2] = gn * n3 - G[2];
  }

  // the raw gradient G of accel() (for callers that add further forces before the projection:
  // the demagnetising field, ss_demag.cuh)
  template <typename Tile, typename P>
  __device__ __forceinline__ static void gradient(const Tile& T, const P& p, real B, real G[3]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const real s1 = (T(c, 0, 1) + T(c, 0, -1)) + (T(c, 1, 0) + T(c, -1, 0));
      const real s2 = (T(c, 0, 2) + T(c, 0, -2)) + (T(c, 2, 0) + T(c, -2, 0));
      G[c] = p.lap2 * s2 + (p.lap0 * T(c, 0, 0) - p.lap1 * s1);
    }
    G[0] += p.dm1 * (T(2, 1, 0) - T(2, -1, 0)) - p.dm2 * (T(2, 2, 0) - T(2, -2, 0));
    G[1] -= p.dm1 * (T(2, 0, 1) - T(2, 0, -1)) - p.dm2 * (T(2, 0, 2) - T(2, 0, -2));
    G[2] += p.dm1 * ((T(1, 0, 1) - T(1, 0, -1)) - (T(0, 1, 0) - T(0, -1, 0))) -
            p.dm2 * ((T(1, 0, 2) - T(1, 0, -2)) - (T(0, 2, 0) - T(0, -2, 0)));
    G[2] -= B + p.K2 * T(2, 0, 0);
  }

  // accel + site-form energy density + charge density of a site whose neighbours are all
  // interior (weights 1): the eq. (1) numerators d_x n, d_y n are formed once and serve the DMI
  // force, the DMI energy kappa n.(curl_h n) and the charge; the exchange energy keeps the
  // plain |n_i - n_j|^2 form (valid for non-unit fields), summed per neighbour shell.
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel_densities_bulk(const Tile& T, const P& p, real B,
                                                              real a[3], real& e, real& q) {
    const real n[3] = {T(0, 0, 0), T(1, 0, 0), T(2, 0, 0)};
    real G[3], dx[3], dy[3];
    real sA0 = real(0), sA1 = real(0), sB0 = real(0), sB1 = real(0);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const real xp1 = T(c, 0, 1), xm1 = T(c, 0, -1), yp1 = T(c, 1, 0), ym1 = T(c, -1, 0);
      const real xp2 = T(c, 0, 2), xm2 = T(c, 0, -2), yp2 = T(c, 2, 0), ym2 = T(c, -2, 0);
      const real s1 = (xp1 + xm1) + (yp1 + ym1);
      const real s2 = (xp2 + xm2) + (yp2 + ym2);
      G[c] = p.lap2 * s2 + (p.lap0 * n[c] - p.lap1 * s1);
      dx[c] = real(8) * (xp1 - xm1) - (xp2 - xm2);
      dy[c] = real(8) * (yp1 - ym1) - (yp2 - ym2);
      real d;
      d = n[c] - xp1; sA0 += d * d;
      d = n[c] - xm1; sA1 += d * d;
      d = n[c] - yp1; sA0 += d * d;
      d = n[c] - ym1; sA1 += d * d;
      d = n[c] - xp2; sB0 += d * d;
      d = n[c] - xm2; sB1 += d * d;
      d = n[c] - yp2; sB0 += d * d;
      d = n[c] - ym2; sB1 += d * d;
    }
    G[0] += p.dm2 * dy[2];
    G[1] -= p.dm2 * dx[2];
    G[2] += p.dm2 * (dx[1] - dy[0]) - (B + p.K2 * n[2]);
    const real gn = (G[0] * n[0] + G[1] * n[1]) + G[2] * n[2];
    a[0] = gn * n[0] - G[0];
    a[1] = gn * n[1] - G[1];
    a[2] = gn * n[2] - G[2];
    const real curl = (n[2] * dx[1] - n[1] * dx[2]) + (n[0] * dy[2] - n[2] * dy[0]);
    e = (p.jA * (sA0 + sA1) + p.jB * (sB0 + sB1)) + p.hk * curl +
        (B * (real(1) - n[2]) + p.K * (real(1) - n[2] * n[2]));
    const real c1 = dx[1] * dy[2] - dx[2] * dy[1], c2 = dx[2] * dy[0] - dx[0] * dy[2],
               c3 = dx[0] * dy[1] - dx[1] * dy[0];
    q = p.qs * ((n[0] * c1 + n[1] * c2) + n[2] * c3);
  }

  // site-form energy density and charge density at an interior site
  template <typename Tile, typename P, typename W>
  __device__ __forceinline__ static void densities(const Tile& T, const P& p, real B,
                                                   const W& w, real& e, real& q) {
    const real n1 = T(0, 0, 0), n2 = T(1, 0, 0), n3 = T(2, 0, 0);
    const int ks[4] = {1, -1, 2, -2};
    const real J4[4] = {real(4) * p.i12h2, real(4) * p.i12h2, real(-0.25) * p.i12h2,
                        real(-0.25) * p.i12h2};  // J_|k| / (4 h^2)
    const real ck[4] = {real(8) * p.i12h, real(-8) * p.i12h, -p.i12h, p.i12h};
    real acc = real(0);
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      {  // x neighbour
        const real m1 = T(0, 0, ks[s]), m2 = T(1, 0, ks[s]), m3 = T(2, 0, ks[s]);
        const real d1 = n1 - m1, d2 = n2 - m2, d3 = n3 - m3;
        const real ex = J4[s] * (d1 * d1 + d2 * d2 + d3 * d3);
        const real cr = n3 * m2 - n2 * m3;  // n_i . (e_x x n_j)
        acc += real(w.wx(s)) * (ex + p.kappa * ck[s] * cr);
      }
      {  // y neighbour
        const real m1 = T(0, ks[s], 0), m2 = T(1, ks[s], 0), m3 = T(2, ks[s], 0);
        const real d1 = n1 - m1, d2 = n2 - m2, d3 = n3 - m3;
        const real ex = J4[s] * (d1 * d1 + d2 * d2 + d3 * d3);
        const real cr = n1 * m3 - n3 * m1;  // n_i . (e_y x n_j)
        acc += real(w.wy(s)) * (ex + p.kappa * ck[s] * cr);
      }
    }
    e = acc + B * (real(1) - n3) + p.K * (real(1) - n3 * n3);
    // q = (1/4pi) n . (Dx n x Dy n)
    const real x1 = Dxn<real>(T, 0), x2 = Dxn<real>(T, 1), x3 = Dxn<real>(T, 2);
    const real y1 = Dyn<real>(T, 0), y2 = Dyn<real>(T, 1), y3 = Dyn<real>(T, 2);
    const real c1 = x2 * y3 - x3 * y2, c2 = x3 * y1 - x1 * y3, c3 = x1 * y2 - x2 * y1;
    q = real(0.07957747154594767) * (p.i12h * p.i12h) * ((n1 * c1 + n2 * c2) + n3 * c3);
  }

  // R(m) = m / |m|
  __device__ __forceinline__ static void project_field(real m[3]) {
    const real r = rsqrt_<real>((m[0] * m[0] + m[1] * m[1]) + m[2] * m[2]);
    m[0] *= r; m[1] *= r; m[2] *= r;
  }
  // v <- u - (u.n) n
  __device__ __forceinline__ static void project_velocity(real u[3], const real n[3]) {
    const real un = (u[0] * n[0] + u[1] * n[1]) + u[2] * n[2];
    u[0] -= un * n[0]; u[1] -= un * n[1]; u[2] -= un * n[2];
  }
};

// ------------------------------------------- chiral magnet with a general DMI table
// e_DMI = kappa sum_mu d_mu . (n x D_mu n)  (eq. (5); DESIGN R16); p.dk[0..2],
// p.dk[3..5] = kappa/(12h) * (d_x, d_y).  Exchange, Zeeman, anisotropy, charge as in CM.
template <typename real>
struct CMG {
  static constexpr int C = 3;

  // weighted eq. (1) numerators of all three components: sum_k w_k (12h c_k) n(i + k mu)
  template <typename Tile, typename W>
  __device__ __forceinline__ static void numerators(const Tile& T, const W& w, real dx[3],
                                                    real dy[3]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      dx[c] = real(8) * (real(w.wx(0)) * T(c, 0, 1) - real(w.wx(1)) * T(c, 0, -1)) -
              (real(w.wx(2)) * T(c, 0, 2) - real(w.wx(3)) * T(c, 0, -2));
      dy[c] = real(8) * (real(w.wy(0)) * T(c, 1, 0) - real(w.wy(1)) * T(c, -1, 0)) -
              (real(w.wy(2)) * T(c, 2, 0) - real(w.wy(3)) * T(c, -2, 0));
    }
  }

  // G = -(Lx+Ly) n + 2 kappa sum_mu (D_mu n) x d_mu - (B + 2K n3) e3 ;  a = -(G - (G.n) n)
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel_from(const Tile& T, const P& p, real B,
                                                    const real dx[3], const real dy[3], real a[3]) {
    const real n[3] = {T(0, 0, 0), T(1, 0, 0), T(2, 0, 0)};
    real G[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const real s1 = (T(c, 0, 1) + T(c, 0, -1)) + (T(c, 1, 0) + T(c, -1, 0));
      const real s2 = (T(c, 0, 2) + T(c, 0, -2)) + (T(c, 2, 0) + T(c, -2, 0));
      G[c] = p.lap2 * s2 + (p.lap0 * n[c] - p.lap1 * s1);
    }
    const auto* kx = p.dk;
    const auto* ky = p.dk + 3;
    G[0] += real(2) * ((dx[1] * kx[2] - dx[2] * kx[1]) + (dy[1] * ky[2] - dy[2] * ky[1]));
    G[1] += real(2) * ((dx[2] * kx[0] - dx[0] * kx[2]) + (dy[2] * ky[0] - dy[0] * ky[2]));
    G[2] += real(2) * ((dx[0] * kx[1] - dx[1] * kx[0]) + (dy[0] * ky[1] - dy[1] * ky[0]));
    G[2] -= B + p.K2 * n[2];
    const real gn = (G[0] * n[0] + G[1] * n[1]) + G[2] * n[2];
    a[0] = gn * n[0] - G[0];
    a[1] = gn * n[1] - G[1];
    a[2] = gn * n[2] - G[2];
  }
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel(const Tile& T, const P& p, real B, real a[3]) {
    real dx[3], dy[3];
    numerators(T, BulkW(), dx, dy);
    accel_from(T, p, B, dx, dy, a);
  }
  // the raw gradient G of accel()
  template <typename Tile, typename P>
  __device__ __forceinline__ static void gradient(const Tile& T, const P& p, real B, real G[3]) {
    real dx[3], dy[3];
    numerators(T, BulkW(), dx, dy);
    const real n2 = T(2, 0, 0);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const real s1 = (T(c, 0, 1) + T(c, 0, -1)) + (T(c, 1, 0) + T(c, -1, 0));
      const real s2 = (T(c, 0, 2) + T(c, 0, -2)) + (T(c, 2, 0) + T(c, -2, 0));
      G[c] = p.lap2 * s2 + (p.lap0 * T(c, 0, 0) - p.lap1 * s1);
    }
    const auto* kx = p.dk;
    const auto* ky = p.dk + 3;
    G[0] += real(2) * ((dx[1] * kx[2] - dx[2] * kx[1]) + (dy[1] * ky[2] - dy[2] * ky[1]));
    G[1] += real(2) * ((dx[2] * kx[0] - dx[0] * kx[2]) + (dy[2] * ky[0] - dy[0] * ky[2]));
    G[2] += real(2) * ((dx[0] * kx[1] - dx[1] * kx[0]) + (dy[0] * ky[1] - dy[1] * ky[0]));
    G[2] -= B + p.K2 * n2;
  }

  // site-form energy and charge densities; wdx, wdy = the WEIGHTED numerators (halo rule R3)
  template <typename Tile, typename P, typename W>
  __device__ __forceinline__ static void densities_from(const Tile& T, const P& p, real B,
                                                        const W& w, const real wdx[3],
                                                        const real wdy[3], const real dx[3],
                                                        const real dy[3], real& e, real& q) {
    const real n[3] = {T(0, 0, 0), T(1, 0, 0), T(2, 0, 0)};
    const int ks[4] = {1, -1, 2, -2};
    real sA = real(0), sB = real(0);
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      real tx = real(0), ty = real(0);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const real ax = n[c] - T(c, 0, ks[s]), ay = n[c] - T(c, ks[s], 0);
        tx += ax * ax;
        ty += ay * ay;
      }
      const real t = real(w.wx(s)) * tx + real(w.wy(s)) * ty;
      if (s < 2) sA += t; else sB += t;
    }
    const auto* kx = p.dk;
    const auto* ky = p.dk + 3;
    // kappa sum_mu d_mu . (n x D_mu n)
    const real dmi =
        (kx[0] * (n[1] * wdx[2] - n[2] * wdx[1]) + kx[1] * (n[2] * wdx[0] - n[0] * wdx[2]) +
         kx[2] * (n[0] * wdx[1] - n[1] * wdx[0])) +
        (ky[0] * (n[1] * wdy[2] - n[2] * wdy[1]) + ky[1] * (n[2] * wdy[0] - n[0] * wdy[2]) +
         ky[2] * (n[0] * wdy[1] - n[1] * wdy[0]));
    e = (p.jA * sA + p.jB * sB) + dmi + (B * (real(1) - n[2]) + p.K * (real(1) - n[2] * n[2]));
    const real c1 = dx[1] * dy[2] - dx[2] * dy[1], c2 = dx[2] * dy[0] - dx[0] * dy[2],
               c3 = dx[0] * dy[1] - dx[1] * dy[0];
    q = p.qs * ((n[0] * c1 + n[1] * c2) + n[2] * c3);
  }
  template <typename Tile, typename P, typename W>
  __device__ __forceinline__ static void densities(const Tile& T, const P& p, real B, const W& w,
                                                   real& e, real& q) {
    real dx[3], dy[3], wdx[3], wdy[3];
    numerators(T, BulkW(), dx, dy);
    numerators(T, w, wdx, wdy);
    densities_from(T, p, B, w, wdx, wdy, dx, dy, e, q);
  }
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel_densities_bulk(const Tile& T, const P& p, real B,
                                                              real a[3], real& e, real& q) {
    real dx[3], dy[3];
    numerators(T, BulkW(), dx, dy);
    accel_from(T, p, B, dx, dy, a);
    densities_from(T, p, B, BulkW(), dx, dy, dx, dy, e, q);
  }

  __device__ __forceinline__ static void project_field(real m[3]) { CM<real>::project_field(m); }
  __device__ __forceinline__ static void project_velocity(real u[3], const real n[3]) {
    CM<real>::project_velocity(u, n);
  }
};

// ------------------------------------------------------------------ abelian Higgs
template <typename real>
struct AH {
  static constexpr int C = 4;  // 0: Re phi, 1: Im phi, 2: A1, 3: A2

  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel(const Tile& T, const P& p, real B, real a[4]) {
    accel_xy(T, p, B, Dxyn<real>(T, 2), Dxyn<real>(T, 3), a);
  }
  // xyA1, xyA2 = (12h)^2 DxDy A1, A2 at the site, supplied by the caller (the flow kernels form
  // them as D_y of per-row D_x values shared by the vertically adjacent sites of a thread)
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel_xy(const Tile& T, const P& p, real, real xyA1,
                                                  real xyA2, real a[4]) {
    const real p1 = T(0, 0, 0), p2 = T(1, 0, 0), A1 = T(2, 0, 0), A2 = T(3, 0, 0);
    const real rho = p1 * p1 + p2 * p2, AA = A1 * A1 + A2 * A2;
    // S_mu,c = 12h * sum_k c_k (A_mu(i+k) + A_mu(i)) phi_c(i+k)
    real Sx1, Sx2, Sy1, Sy2;
    {
      const real am2 = T(2, 0, -2) + A1, am1 = T(2, 0, -1) + A1, ap1 = T(2, 0, 1) + A1,
                 ap2 = T(2, 0, 2) + A1;
      Sx1 = d1n<real>(am2 * T(0, 0, -2), am1 * T(0, 0, -1), ap1 * T(0, 0, 1), ap2 * T(0, 0, 2));
      Sx2 = d1n<real>(am2 * T(1, 0, -2), am1 * T(1, 0, -1), ap1 * T(1, 0, 1), ap2 * T(1, 0, 2));
    }
    {
      const real am2 = T(3, -2, 0) + A2, am1 = T(3, -1, 0) + A2, ap1 = T(3, 1, 0) + A2,
                 ap2 = T(3, 2, 0) + A2;
      Sy1 = d1n<real>(am2 * T(0, -2, 0), am1 * T(0, -1, 0), ap1 * T(0, 1, 0), ap2 * T(0, 2, 0));
      Sy2 = d1n<real>(am2 * T(1, -2, 0), am1 * T(1, -1, 0), ap1 * T(1, 1, 0), ap2 * T(1, 2, 0));
    }
    const real pot = real(0.5) * p.lambda * (real(1) - rho);
    const real G1 = -(Lxn<real>(T, 0) + Lyn<real>(T, 0)) * p.i12h2 - (Sx2 + Sy2) * p.i12h +
                    (AA - pot) * p1;
    const real G2 = -(Lxn<real>(T, 1) + Lyn<real>(T, 1)) * p.i12h2 + (Sx1 + Sy1) * p.i12h +
                    (AA - pot) * p2;
    const real ii = p.i12h * p.i12h;
    const real G3 = -Lyn<real>(T, 2) * p.i12h2 + xyA2 * ii +
                    (p2 * Dxn<real>(T, 0) - p1 * Dxn<real>(T, 1)) * p.i12h + A1 * rho;
    const real G4 = -Lxn<real>(T, 3) * p.i12h2 + xyA1 * ii +
                    (p2 * Dyn<real>(T, 0) - p1 * Dyn<real>(T, 1)) * p.i12h + A2 * rho;
    a[0] = -G1; a[1] = -G2; a[2] = -G3; a[3] = -G4;
  }

  template <typename Tile, typename P, typename W>
  __device__ __forceinline__ static void densities(const Tile& T, const P& p, real,
                                                   const W& w, real& e, real& q) {
    const real p1 = T(0, 0, 0), p2 = T(1, 0, 0), A1 = T(2, 0, 0), A2 = T(3, 0, 0);
    const real rho = p1 * p1 + p2 * p2;
    const int ks[4] = {1, -1, 2, -2};
    const real J4[4] = {real(4) * p.i12h2, real(4) * p.i12h2, real(-0.25) * p.i12h2,
                        real(-0.25) * p.i12h2};
    const real ck[4] = {real(8) * p.i12h, real(-8) * p.i12h, -p.i12h, p.i12h};
    real acc = real(0.5) * (A1 * A1 + A2 * A2) * rho +
               real(0.125) * p.lambda * (real(1) - rho) * (real(1) - rho);
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      {  // x bond: A_mu = A1, transverse A2
        const real q1 = T(0, 0, ks[s]), q2 = T(1, 0, ks[s]);
        const real d1 = p1 - q1, d2 = p2 - q2, dA = A2 - T(3, 0, ks[s]);
        const real im = p1 * q2 - p2 * q1;
        acc += real(w.wx(s)) * (J4[s] * (d1 * d1 + d2 * d2) -
                               real(0.5) * ck[s] * (A1 + T(2, 0, ks[s])) * im + J4[s] * (dA * dA));
      }
      {  // y bond: A_mu = A2, transverse A1
        const real q1 = T(0, ks[s], 0), q2 = T(1, ks[s], 0);
        const real d1 = p1 - q1, d2 = p2 - q2, dA = A1 - T(2, ks[s], 0);
        const real im = p1 * q2 - p2 * q1;
        acc += real(w.wy(s)) * (J4[s] * (d1 * d1 + d2 * d2) -
                               real(0.5) * ck[s] * (A2 + T(3, ks[s], 0)) * im + J4[s] * (dA * dA));
      }
    }
    // mixed term: + 1/2 [ A2 Wxy(A1) + A1 Wxy(A2) ], Wxy = weighted DxDy over corner sites
    real W1 = real(0), W2 = real(0);
#pragma unroll
    for (int sk = 0; sk < 4; ++sk)
#pragma unroll
      for (int sl = 0; sl < 4; ++sl) {
        const real wt = (w.wx(sk) == 1 && w.wy(sl) == 1) ? real(1) : real(2);
        const real cc = ck[sk] * ck[sl] * wt;
        W1 += cc * T(2, ks[sl], ks[sk]);
        W2 += cc * T(3, ks[sl], ks[sk]);
      }
    e = acc + real(0.5) * (A2 * W1 + A1 * W2);
    q = real(0.15915494309189535) * p.i12h * (Dxn<real>(T, 3) - Dyn<real>(T, 2));
  }

  // accel + site-form energy density + flux density of a site whose neighbours are all interior:
  // the bond term -1/2 c_k (A_i + A_j) Im(phi_i* phi_j) is p1 S_2 - p2 S_1 with the sums
  // S_mu,c = sum_k c_k (A_mu,i + A_mu,j) phi_c,j of the force, and the mixed term is
  // 1/2 (A2 DxDy A1 + A1 DxDy A2) with the corner sums of the force.
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel_densities_bulk(const Tile& T, const P& p, real B,
                                                              real a[4], real& e, real& q) {
    accel_densities_bulk_xy(T, p, B, Dxyn<real>(T, 2), Dxyn<real>(T, 3), a, e, q);
  }
  template <typename Tile, typename P>
  __device__ __forceinline__ static void accel_densities_bulk_xy(const Tile& T, const P& p, real,
                                                                 real xyA1, real xyA2, real a[4],
                                                                 real& e, real& q) {
    const real p1 = T(0, 0, 0), p2 = T(1, 0, 0), A1 = T(2, 0, 0), A2 = T(3, 0, 0);
    const real rho = p1 * p1 + p2 * p2, AA = A1 * A1 + A2 * A2;
    real Sx1, Sx2, Sy1, Sy2;
    {
      const real am2 = T(2, 0, -2) + A1, am1 = T(2, 0, -1) + A1, ap1 = T(2, 0, 1) + A1,
                 ap2 = T(2, 0, 2) + A1;
      Sx1 = d1n<real>(am2 * T(0, 0, -2), am1 * T(0, 0, -1), ap1 * T(0, 0, 1), ap2 * T(0, 0, 2));
      Sx2 = d1n<real>(am2 * T(1, 0, -2), am1 * T(1, 0, -1), ap1 * T(1, 0, 1), ap2 * T(1, 0, 2));
    }
    {
      const real am2 = T(3, -2, 0) + A2, am1 = T(3, -1, 0) + A2, ap1 = T(3, 1, 0) + A2,
                 ap2 = T(3, 2, 0) + A2;
      Sy1 = d1n<real>(am2 * T(0, -2, 0), am1 * T(0, -1, 0), ap1 * T(0, 1, 0), ap2 * T(0, 2, 0));
      Sy2 = d1n<real>(am2 * T(1, -2, 0), am1 * T(1, -1, 0), ap1 * T(1, 1, 0), ap2 * T(1, 2, 0));
    }
    const real pot = real(0.5) * p.lambda * (real(1) - rho);
    const real G1 = -(Lxn<real>(T, 0) + Lyn<real>(T, 0)) * p.i12h2 - (Sx2 + Sy2) * p.i12h +
                    (AA - pot) * p1;
    const real G2 = -(Lxn<real>(T, 1) + Lyn<real>(T, 1)) * p.i12h2 + (Sx1 + Sy1) * p.i12h +
                    (AA - pot) * p2;
    const real ii = p.i12h * p.i12h;
    const real dxA2 = Dxn<real>(T, 3), dyA1 = Dyn<real>(T, 2);
    const real G3 = -Lyn<real>(T, 2) * p.i12h2 + xyA2 * ii +
                    (p2 * Dxn<real>(T, 0) - p1 * Dxn<real>(T, 1)) * p.i12h + A1 * rho;
    const real G4 = -Lxn<real>(T, 3) * p.i12h2 + xyA1 * ii +
                    (p2 * Dyn<real>(T, 0) - p1 * Dyn<real>(T, 1)) * p.i12h + A2 * rho;
    a[0] = -G1; a[1] = -G2; a[2] = -G3; a[3] = -G4;
    // bond sums per neighbour shell: |phi_i - phi_j|^2 + (transverse A_i - A_j)^2
    real sA = real(0), sB = real(0);
    const int ks[4] = {1, -1, 2, -2};
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const real dx1 = p1 - T(0, 0, ks[s]), dx2 = p2 - T(1, 0, ks[s]), dxa = A2 - T(3, 0, ks[s]);
      const real dy1 = p1 - T(0, ks[s], 0), dy2 = p2 - T(1, ks[s], 0), dya = A1 - T(2, ks[s], 0);
      const real t = ((dx1 * dx1 + dx2 * dx2) + dxa * dxa) + ((dy1 * dy1 + dy2 * dy2) + dya * dya);
      if (s < 2) sA += t; else sB += t;
    }
    e = (real(0.5) * AA * rho + real(0.125) * p.lambda * (real(1) - rho) * (real(1) - rho)) +
        (p.jA * sA + p.jB * sB) -
        real(0.5) * p.i12h * (p1 * (Sx2 + Sy2) - p2 * (Sx1 + Sy1)) +
        real(0.5) * ii * (A2 * xyA1 + A1 * xyA2);
    q = real(0.15915494309189535) * p.i12h * (dxA2 - dyA1);
  }

  __device__ __forceinline__ static void project_field(real*) {}
  __device__ __forceinline__ static void project_velocity(real*, const real*) {}
};

// ------------------------------------------------------------------ baby Skyrme
// E = 1/2 |grad m|^2 + (kappa^2/2) |D_x m x D_y m|^2 + V(m), m in S^2 (PAPER.md:323 Table 2, :90;
// DESIGN R18).  Dirichlet term as the chiral magnet's exchange (bond form, halo weights R3);
// Skyrme term and potential are site sums over the interior with eq. (1).  Exact gradient in flux
// form: a = D_x m, b = D_y m, w = a x b, F_x = kappa^2 (b x w), F_y = kappa^2 (w x a) (0 on the
// halo), G = -(Lx + Ly) m - D_x F_x - D_y F_y + dV/dm -- radius 4, evaluated by the tile kernels
// of ss_bs.cuh in two passes.  p supplies i12h, jA, jB, bs_k2 = kappa^2, bs_mu2, bs_pot, bs_potN.
template <typename real>
struct BS {
  static constexpr int C = 3;
  static constexpr int POT_STANDARD = 0, POT_EASY_PLANE = 1, POT_BROKEN = 2;

  __device__ __forceinline__ static void cpow(real x, real y, int N, real& re, real& im) {
    real a = real(1), b = real(0);
    for (int k = 0; k < N; ++k) {
      const real t = a * x - b * y;
      b = a * y + b * x;
      a = t;
    }
    re = a;
    im = b;
  }
  // standard mu^2 (1 - m3); easy plane 1/2 mu^2 m1^2; broken mu^2 |1 - (m1 + i m2)^N|^2 (1 - m3)
  template <typename P>
  __device__ __forceinline__ static real potential(const P& p, real m1, real m2, real m3) {
    if (p.bs_pot == POT_STANDARD) return p.bs_mu2 * (real(1) - m3);
    if (p.bs_pot == POT_EASY_PLANE) return real(0.5) * p.bs_mu2 * (m1 * m1);
    real a, b;
    cpow(m1, m2, p.bs_potN, a, b);
    return p.bs_mu2 * ((real(1) - a) * (real(1) - a) + b * b) * (real(1) - m3);
  }
  template <typename P>
  __device__ __forceinline__ static void potential_grad(const P& p, real m1, real m2, real m3,
                                                        real dV[3]) {
    if (p.bs_pot == POT_STANDARD) { dV[0] = real(0); dV[1] = real(0); dV[2] = -p.bs_mu2; return; }
    if (p.bs_pot == POT_EASY_PLANE) { dV[0] = p.bs_mu2 * m1; dV[1] = real(0); dV[2] = real(0); return; }
    real a, b, c, d;
    const real N = real(p.bs_potN);
    cpow(m1, m2, p.bs_potN, a, b);
    cpow(m1, m2, p.bs_potN - 1, c, d);
    const real P2 = (real(1) - a) * (real(1) - a) + b * b;
    dV[0] = p.bs_mu2 * (real(1) - m3) * (real(2) * N * (b * d - (real(1) - a) * c));
    dV[1] = p.bs_mu2 * (real(1) - m3) * (real(2) * N * ((real(1) - a) * d + b * c));
    dV[2] = -p.bs_mu2 * P2;
  }
  // a = D_x m, b = D_y m, w = a x b at the site
  template <typename Tile, typename P>
  __device__ __forceinline__ static void derivs(const Tile& T, const P& p, real a[3], real b[3],
                                                real w[3]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      a[c] = p.i12h * Dxn<real>(T, c);
      b[c] = p.i12h * Dyn<real>(T, c);
    }
    w[0] = a[1] * b[2] - a[2] * b[1];
    w[1] = a[2] * b[0] - a[0] * b[2];
    w[2] = a[0] * b[1] - a[1] * b[0];
  }
  template <typename P>
  __device__ __forceinline__ static void flux(const P& p, const real a[3], const real b[3],
                                              const real w[3], real Fx[3], real Fy[3]) {
    Fx[0] = p.bs_k2 * (b[1] * w[2] - b[2] * w[1]);
    Fx[1] = p.bs_k2 * (b[2] * w[0] - b[0] * w[2]);
    Fx[2] = p.bs_k2 * (b[0] * w[1] - b[1] * w[0]);
    Fy[0] = p.bs_k2 * (w[1] * a[2] - w[2] * a[1]);
    Fy[1] = p.bs_k2 * (w[2] * a[0] - w[0] * a[2]);
    Fy[2] = p.bs_k2 * (w[0] * a[1] - w[1] * a[0]);
  }
  // site-form energy density and degree density from w = D_x m x D_y m
  template <typename Tile, typename P, typename W>
  __device__ __forceinline__ static void densities_w(const Tile& T, const P& p, const W& wt,
                                                     const real w[3], real& e, real& q) {
    const real m[3] = {T(0, 0, 0), T(1, 0, 0), T(2, 0, 0)};
    const int ks[4] = {1, -1, 2, -2};
    real sA = real(0), sB = real(0);
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      real tx = real(0), ty = real(0);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const real ax = m[c] - T(c, 0, ks[s]), ay = m[c] - T(c, ks[s], 0);
        tx += ax * ax;
        ty += ay * ay;
      }
      const real t = real(wt.wx(s)) * tx + real(wt.wy(s)) * ty;
      if (s < 2) sA += t; else sB += t;
    }
    e = (p.jA * sA + p.jB * sB) +
        real(0.5) * p.bs_k2 * ((w[0] * w[0] + w[1] * w[1]) + w[2] * w[2]) +
        potential(p, m[0], m[1], m[2]);
    q = real(0.07957747154594767) * ((m[0] * w[0] + m[1] * w[1]) + m[2] * w[2]);
  }
  template <typename Tile, typename P, typename W>
  __device__ __forceinline__ static void densities(const Tile& T, const P& p, real, const W& wt,
                                                   real& e, real& q) {
    real a[3], b[3], w[3];
    derivs(T, p, a, b, w);
    densities_w(T, p, wt, w, e, q);
  }
  __device__ __forceinline__ static void project_field(real m[3]) { CM<real>::project_field(m); }
  __device__ __forceinline__ static void project_velocity(real u[3], const real n[3]) {
    CM<real>::project_velocity(u, n);
  }
};

template <int THEORY, typename real> struct TheoryOf;
template <typename real> struct TheoryOf<kCM, real> { using type = CM<real>; };
template <typename real> struct TheoryOf<kAH, real> { using type = AH<real>; };
template <typename real> struct TheoryOf<kCMG, real> { using type = CMG<real>; };
template <typename real> struct TheoryOf<kBS, real> { using type = BS<real>; };

}  // namespace ss
