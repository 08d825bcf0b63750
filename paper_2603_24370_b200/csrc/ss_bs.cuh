// Baby-Skyrme flow step (PAPER.md:323 Table 2, :90; DESIGN R18; SURVEY 8(f) NEXT-2b): one tile
// kernel per RK4 stage.  The exact gradient of the Skyrme term has radius 4 (the flux
// F_mu = d e4 / d(D_mu m) needs radius 2, its divergence radius 2 again), so a tile of 64 x 16
// output sites stages its field on 72 x 24 sites and evaluates in two passes through shared memory:
//
//   bs_stage_kernel<real, STAGE>
//     phase 1  stage field psi = R(phi + alpha*vh + beta*a_prev) on the tile + 4 sites of halo,
//              rebuilt from phi, v, a_prev (never stored in HBM)                         -> smem
//     phase 2  a = D_x psi, b = D_y psi, w = a x b, F_x = kappa^2 b x w, F_y = kappa^2 w x a at the
//              tile + 2 sites in x (F_x) and in y (F_y); F = 0 on the frozen halo         -> smem
//     phase 3  G = -(Lx + Ly) psi - D_x F_x - D_y F_y + dV/dm, acceleration -Pi G
//       STAGE 1: psi = phi; also site energy / degree densities -> row-segment partial sums
//       STAGE 4: + RK4 combine, projections (PAPER.md:129+154), KE partial sums, writes the new
//                (phi, v) into the other ping-pong buffer
//       STAGE 5: the whole one-gradient-per-step (velocity Verlet, DESIGN R15) step: psi = phi_new
//                = R(phi + dt (vh + dt/2 a)), a_new = -Pi G(phi_new), v_new = Pi(vh + dt/2 a +
//                dt/2 a_new), e, q, KE partial sums; writes phi_new, v_new, a_new
//
// Algorithmic bytes: stage 2 reads phi, v, writes a2 (3 C R); stage 3 reads phi, v, a1, writes a3
// (4); stage 4 reads phi, v, a1, a2, a3, writes phi', v' (7); stage 1 reads phi', writes a1 (2):
// 16 C R per site-step.  The arrest decision exists before stage 2 starts (no speculation).
#pragma once
#include "ss_theory.cuh"

namespace ss {

constexpr int BTX = SEG, BTY = 16;                     // output sites of a tile
constexpr int BH = 2 * HALO;                           // halo of the stage-field tile
constexpr int BMX = BTX + 2 * BH, BMY = BTY + 2 * BH;  // 72 x 24
constexpr int BFXW = BTX + 2 * HALO;                   // F_x lives on 68 x 16
constexpr int BFYH = BTY + 2 * HALO;                   // F_y lives on 64 x 20
constexpr int BBX = 64, BBY = 4;                       // threads

template <typename real>
struct BsArgs {
  const real* phi;    // [batch][3][Ny][Nx] current field (halo frozen)
  const real* vel;    // velocity
  const real* aprev;  // acceleration entering the stage field (a1 for stage 3, a2 for stage 4)
  real* aout;         // acceleration written by stages 1-3
  const real* a1;     // stage 4 only
  const real* a3;     // stage 4 only
  real* phi_out;      // stage 4 only: phi^{n+1}
  real* vel_out;      // stage 4 only: v^{n+1}
  double* part_e;     // [batch][Ny][nseg] row-segment partial sums (stage 1)
  double* part_q;
  double* part_ke;    // (stage 4)
  const LatticeState* state;
  int Nx, Ny, nseg;
  long long plane;    // Nx*Ny
  real alpha, beta;   // stage field = R(phi + alpha*vh + beta*aprev)
  real dt, sdt2, sdt; // dt, dt^2/6, dt/6
  real i12h, i12h2;   // 1/(12h), 1/(12h^2)
  real lap0, lap1, lap2;  // 60, 16, 1 / (12 h^2)
  real jA, jB;            // J1/4h^2, J2/4h^2
  real bs_k2, bs_mu2;     // kappa^2, mu^2
  int bs_pot, bs_potN;
};

template <typename real>
struct BsSmem {
  real m[3][BMY][BMX];
  real fx[3][BTY][BFXW];
  real fy[3][BFYH][BTX];
};

template <typename real, int STAGE>
__global__ void __launch_bounds__(BBX* BBY, 2) bs_stage_kernel(const __grid_constant__ BsArgs<real> p) {
  using Th = BS<real>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  BsSmem<real>& sm = *reinterpret_cast<BsSmem<real>*>(smem_raw);
  __shared__ double red[3][BTY][BBX / 32];

  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z;
  const int x0 = blockIdx.x * BTX, y0 = blockIdx.y * BTY;
  const long long lat = (long long)b * 3 * p.plane;
  const real* __restrict__ phi = p.phi + lat;
  const real* __restrict__ vel = p.vel + lat;
  const real* __restrict__ aprev = p.aprev + lat;
  const int tid = threadIdx.y * BBX + threadIdx.x;
  const bool vz = (STAGE > 1) ? (p.state[b].v_is_zero != 0) : true;
  auto interior = [&](int gx, int gy) {
    return gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO;
  };

  // ---- phase 1: stage field on the tile + 4.  A thread owns NS1 sites; all loads of one input
  // array are issued before any is used (27 independent loads in flight per thread and array:
  // the tile is read at L2 latency once, not once per site)
  constexpr int NS1 = (BMY * BMX + BBX * BBY - 1) / (BBX * BBY);
  {
    long long off[NS1];
    bool in[NS1], inter[NS1];
    real m[NS1][3];
#pragma unroll
    for (int k = 0; k < NS1; ++k) {
      const int idx = tid + k * BBX * BBY;
      const int ly = idx / BMX, lx = idx - ly * BMX;
      const int gx = x0 - BH + lx, gy = y0 - BH + ly;
      in[k] = idx < BMY * BMX && gx >= 0 && gx < Nx && gy >= 0 && gy < Ny;
      inter[k] = in[k] && interior(gx, gy);
      off[k] = in[k] ? (long long)gy * Nx + gx : 0;
    }
#pragma unroll
    for (int k = 0; k < NS1; ++k)
#pragma unroll
      for (int c = 0; c < 3; ++c) m[k][c] = in[k] ? phi[c * p.plane + off[k]] : real(0);
    if (STAGE == 5) {  // velocity Verlet (DESIGN R15): phi' = R(phi + dt (vh + dt/2 a))
      real v[NS1][3], ap[NS1][3];
#pragma unroll
      for (int k = 0; k < NS1; ++k)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          v[k][c] = (inter[k] && !vz) ? vel[c * p.plane + off[k]] : real(0);
          ap[k][c] = inter[k] ? aprev[c * p.plane + off[k]] : real(0);
        }
#pragma unroll
      for (int k = 0; k < NS1; ++k) {
#pragma unroll
        for (int c = 0; c < 3; ++c) m[k][c] = m[k][c] + p.dt * (v[k][c] + p.beta * ap[k][c]);
        if (inter[k]) Th::project_field(m[k]);
      }
    } else if (STAGE > 1) {  // halo sites of every stage field are the frozen halo
      if (!vz) {
        real v[NS1][3];
#pragma unroll
        for (int k = 0; k < NS1; ++k)
#pragma unroll
          for (int c = 0; c < 3; ++c) v[k][c] = inter[k] ? vel[c * p.plane + off[k]] : real(0);
#pragma unroll
        for (int k = 0; k < NS1; ++k)
#pragma unroll
          for (int c = 0; c < 3; ++c) m[k][c] = m[k][c] + p.alpha * v[k][c];
      } else {
#pragma unroll
        for (int k = 0; k < NS1; ++k)
#pragma unroll
          for (int c = 0; c < 3; ++c) m[k][c] = m[k][c] + p.alpha * real(0);
      }
      if (STAGE > 2) {
        real ap[NS1][3];
#pragma unroll
        for (int k = 0; k < NS1; ++k)
#pragma unroll
          for (int c = 0; c < 3; ++c) ap[k][c] = inter[k] ? aprev[c * p.plane + off[k]] : real(0);
#pragma unroll
        for (int k = 0; k < NS1; ++k)
#pragma unroll
          for (int c = 0; c < 3; ++c) m[k][c] = m[k][c] + p.beta * ap[k][c];
      }
#pragma unroll
      for (int k = 0; k < NS1; ++k)
        if (inter[k]) Th::project_field(m[k]);
    }
#pragma unroll
    for (int k = 0; k < NS1; ++k) {
      const int idx = tid + k * BBX * BBY;
      if (idx < BMY * BMX) {
        const int ly = idx / BMX, lx = idx - ly * BMX;
#pragma unroll
        for (int c = 0; c < 3; ++c) sm.m[c][ly][lx] = m[k][c];
      }
    }
  }
  __syncthreads();

  // ---- phase 2: fluxes at (fx, fy) relative to the tile origin, fx in [-2, 66), fy in [-2, 18)
  auto flux_site = [&](int fx, int fy) {
    real Fx[3] = {real(0), real(0), real(0)}, Fy[3] = {real(0), real(0), real(0)};
    if (interior(x0 + fx, y0 + fy)) {
      auto T = [&](int c, int dy, int dx) -> real { return sm.m[c][fy + BH + dy][fx + BH + dx]; };
      real a[3], bb[3], w[3];
      Th::derivs(T, p, a, bb, w);
      Th::flux(p, a, bb, w, Fx, Fy);
    }
    if (fy >= 0 && fy < BTY) {
#pragma unroll
      for (int c = 0; c < 3; ++c) sm.fx[c][fy][fx + HALO] = Fx[c];
    }
    if (fx >= 0 && fx < BTX) {
#pragma unroll
      for (int c = 0; c < 3; ++c) sm.fy[c][fy + HALO][fx] = Fy[c];
    }
  };
#pragma unroll 1
  for (int r = 0; r < BFYH / BBY; ++r) flux_site(threadIdx.x, r * BBY + threadIdx.y - HALO);
  if (tid < 2 * HALO * BTY) {  // the four x-halo columns of F_x
    const int q = tid % (2 * HALO);
    flux_site(q < HALO ? q - HALO : BTX + q - HALO, tid / (2 * HALO));
  }
  __syncthreads();

  // ---- phase 3
  const int gx = x0 + threadIdx.x;
  const int warp_in_row = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll 1
  for (int r = 0; r < BTY / BBY; ++r) {
    const int ly = r * BBY + threadIdx.y;
    const int gy = y0 + ly;
    const bool active = interior(gx, gy);
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    if (active) {
      const int cx = threadIdx.x + BH, cy = ly + BH;
      auto T = [&](int c, int dy, int dx) -> real { return sm.m[c][cy + dy][cx + dx]; };
      const real m[3] = {T(0, 0, 0), T(1, 0, 0), T(2, 0, 0)};
      real dV[3], G[3];
      Th::potential_grad(p, m[0], m[1], m[2], dV);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const real s1n = (T(c, 0, 1) + T(c, 0, -1)) + (T(c, 1, 0) + T(c, -1, 0));
        const real s2n = (T(c, 0, 2) + T(c, 0, -2)) + (T(c, 2, 0) + T(c, -2, 0));
        const real* fxr = &sm.fx[c][ly][threadIdx.x + HALO];
        const real divx = d1n<real>(fxr[-2], fxr[-1], fxr[1], fxr[2]);
        const real divy = d1n<real>(sm.fy[c][ly][threadIdx.x], sm.fy[c][ly + 1][threadIdx.x],
                                    sm.fy[c][ly + 3][threadIdx.x], sm.fy[c][ly + 4][threadIdx.x]);
        G[c] = (p.lap2 * s2n + (p.lap0 * m[c] - p.lap1 * s1n)) - p.i12h * (divx + divy) + dV[c];
      }
      const real gn = (G[0] * m[0] + G[1] * m[1]) + G[2] * m[2];
      const real a[3] = {gn * m[0] - G[0], gn * m[1] - G[1], gn * m[2] - G[2]};
      const long long o = (long long)gy * Nx + gx;
      if (STAGE != 4) {
#pragma unroll
        for (int c = 0; c < 3; ++c) p.aout[lat + c * p.plane + o] = a[c];
      }
      if (STAGE == 1 || STAGE == 5) {
        real e, q;
        Th::densities(T, p, real(0), EdgeW(gx, gy, Nx, Ny), e, q);
        s0 = double(e);
        s1 = double(q);
      }
      if (STAGE == 5) {  // second half kick with the new acceleration, tangent projection, KE
        real u[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const long long oc = c * p.plane + o;
          const real vh = vz ? real(0) : vel[oc];
          u[c] = (vh + p.beta * aprev[oc]) + p.beta * a[c];
        }
        Th::project_velocity(u, m);
        real v2 = real(0);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          p.phi_out[lat + c * p.plane + o] = m[c];
          p.vel_out[lat + c * p.plane + o] = u[c];
          v2 += u[c] * u[c];
        }
        s2 = 0.5 * double(v2);
      }
      if (STAGE == 4) {
        real f[3], u[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const long long oc = c * p.plane + o;
          const real vh = vz ? real(0) : vel[oc];
          const real A1 = p.a1[lat + oc], A2 = aprev[oc], A3 = p.a3[lat + oc];
          f[c] = (phi[oc] + p.dt * vh) + p.sdt2 * ((A1 + A2) + A3);
          u[c] = vh + p.sdt * ((A1 + real(2) * A2) + (real(2) * A3 + a[c]));
        }
        Th::project_field(f);
        Th::project_velocity(u, f);
        real v2 = real(0);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          p.phi_out[lat + c * p.plane + o] = f[c];
          p.vel_out[lat + c * p.plane + o] = u[c];
          v2 += u[c] * u[c];
        }
        s0 = 0.5 * double(v2);
      }
    }
    if (STAGE == 1 || STAGE >= 4) {  // first five levels of the canonical tree (DESIGN R10)
      s0 = warp_tree(s0);
      if (STAGE != 4) s1 = warp_tree(s1);
      if (STAGE == 5) s2 = warp_tree(s2);
      if (lane == 0) {
        red[0][ly][warp_in_row] = s0;
        if (STAGE != 4) red[1][ly][warp_in_row] = s1;
        if (STAGE == 5) red[2][ly][warp_in_row] = s2;
      }
    }
  }
  if (STAGE == 1 || STAGE >= 4) {
    __syncthreads();
    if (tid < BTY && y0 + tid < Ny) {
      const long long po = ((long long)b * Ny + (y0 + tid)) * p.nseg + blockIdx.x;
      static_assert(BBX / 32 == 2, "row segment = two warps");
      if (STAGE != 4) {
        p.part_e[po] = red[0][tid][0] + red[0][tid][1];
        p.part_q[po] = red[1][tid][0] + red[1][tid][1];
        if (STAGE == 5) p.part_ke[po] = red[2][tid][0] + red[2][tid][1];
      } else {
        p.part_ke[po] = red[0][tid][0] + red[0][tid][1];
      }
    }
  }
}

}  // namespace ss
