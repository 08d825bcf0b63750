// Kernels of the flow step (one launch per RK4 stage + two small reduction kernels).
//
// stage_kernel<THEORY, real, STAGE>   ("derivative ... energy gradient ... Runge-
//   Kutta stages" fused into one pass per stage):
//     phase 1  stage field psi = R(phi + alpha*vhat + beta*aprev) on the tile plus a halo of 2,
//              recomputed from phi, v, a_prev instead of being stored by the previous stage
//              (16*C*sizeof(real) bytes per site-step instead of 21*C*sizeof(real)) -> smem
//     phase 2  a = -Pi_psi G(psi) from smem (eq. 1, 2 stencils)
//       STAGE 1: psi = phi; also energy / charge densities -> row-segment partial sums
//       STAGE 4: + RK4 combine, projections (PAPER.md:129+154), KE partial sums, writes the
//                new (phi, v) into the other ping-pong buffer
// row_reduce_kernel / finalize_kernel: canonical tree (DESIGN R10) + arrest (eq. 4) on device.
#pragma once
#include "ss_theory.cuh"

namespace ss {

constexpr int TX = SEG;  // tile width  = row segment of the reduction tree
constexpr int TY = 16;   // tile height
constexpr int BX = 64, BY = 4;
constexpr int TXP = TX + 2 * HALO, TYP = TY + 2 * HALO;

template <typename real, int C>
struct SmemTile {
  real v[C][TYP][TXP];
};

template <int THEORY, typename real, int STAGE>
__global__ void __launch_bounds__(BX* BY) stage_kernel(const __grid_constant__ StageArgs<real> p) {
  using Th = typename TheoryOf<THEORY, real>::type;
  constexpr int C = Th::C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SmemTile<real, C>& sm = *reinterpret_cast<SmemTile<real, C>*>(smem_raw);
  __shared__ double red[3][TY][BX / 32];

  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const long long lat = (long long)b * C * p.plane;
  const real* __restrict__ phi = p.phi + lat;
  const real* __restrict__ vel = p.vel + lat;
  const real* __restrict__ aprev = p.aprev + lat;
  const int tid = threadIdx.y * BX + threadIdx.x;
  const bool vz = (STAGE > 1) ? (p.state[b].v_is_zero != 0) : true;

  // ---- phase 1: stage field on tile + halo
  for (int idx = tid; idx < TYP * TXP; idx += BX * BY) {
    const int ly = idx / TXP, lx = idx - ly * TXP;
    const int gx = x0 - HALO + lx, gy = y0 - HALO + ly;
    real m[C];
#pragma unroll
    for (int c = 0; c < C; ++c) m[c] = real(0);
    if (gx >= 0 && gx < Nx && gy >= 0 && gy < Ny) {
      const long long o = (long long)gy * Nx + gx;
#pragma unroll
      for (int c = 0; c < C; ++c) m[c] = phi[c * p.plane + o];
      const bool inter = gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO;
      if (STAGE > 1 && inter) {
#pragma unroll
        for (int c = 0; c < C; ++c) {
          const real vh = vz ? real(0) : vel[c * p.plane + o];
          m[c] = m[c] + p.alpha * vh;
          if (STAGE > 2) m[c] = m[c] + p.beta * aprev[c * p.plane + o];
        }
        Th::project_field(m);
      }
    }
#pragma unroll
    for (int c = 0; c < C; ++c) sm.v[c][ly][lx] = m[c];
  }
  __syncthreads();

  // ---- phase 2
  const int gx = x0 + threadIdx.x;
  const real Bz = real(p.Bb[b]);
  const int warp_in_row = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll 1
  for (int r = 0; r < TY / BY; ++r) {
    const int ly = r * BY + threadIdx.y;
    const int gy = y0 + ly;
    const bool active = gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO;
    double s0 = 0.0, s1 = 0.0;
    if (active) {
      const int cx = threadIdx.x + HALO, cy = ly + HALO;
      auto T = [&](int c, int dy, int dx) -> real { return sm.v[c][cy + dy][cx + dx]; };
      real a[C];
      Th::accel(T, p, Bz, a);
      const long long o = (long long)gy * Nx + gx;
      if (STAGE < 4) {
#pragma unroll
        for (int c = 0; c < C; ++c) p.aout[lat + c * p.plane + o] = a[c];
      }
      if (STAGE == 1) {
        real e, q;
        EdgeW w(gx, gy, Nx, Ny);
        Th::densities(T, p, Bz, w, e, q);
        s0 = double(e);
        s1 = double(q);
      }
      if (STAGE == 4) {
        real f[C], u[C];
#pragma unroll
        for (int c = 0; c < C; ++c) {
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
        for (int c = 0; c < C; ++c) {
          p.phi_out[lat + c * p.plane + o] = f[c];
          p.vel_out[lat + c * p.plane + o] = u[c];
          v2 += u[c] * u[c];
        }
        s0 = 0.5 * double(v2);
      }
    }
    if (STAGE == 1 || STAGE == 4) {
      s0 = warp_tree(s0);
      if (STAGE == 1) s1 = warp_tree(s1);
      if (lane == 0) {
        red[0][ly][warp_in_row] = s0;
        if (STAGE == 1) red[1][ly][warp_in_row] = s1;
      }
    }
  }
  if (STAGE == 1 || STAGE == 4) {
    __syncthreads();
    if (tid < TY && y0 + tid < Ny) {
      const long long po = ((long long)b * Ny + (y0 + tid)) * p.nseg + blockIdx.x;
      static_assert(BX / 32 == 2, "row segment = two warps");
      if (STAGE == 1) {
        p.part_e[po] = red[0][tid][0] + red[0][tid][1];
        p.part_q[po] = red[1][tid][0] + red[1][tid][1];
      } else {
        p.part_ke[po] = red[0][tid][0] + red[0][tid][1];
      }
    }
  }
}

// In-thread aligned pairwise tree over m (power of two, <= 32) consecutive values.
__device__ __forceinline__ double chunk_tree(const double* src, long long first, long long n, int m) {
  double t[32];
#pragma unroll 1
  for (int i = 0; i < m; ++i) t[i] = (first + i < n) ? src[first + i] : 0.0;
#pragma unroll 1
  for (int s = m; s > 1; s >>= 1)
#pragma unroll 1
    for (int i = 0; i < s / 2; ++i) t[i] = t[2 * i] + t[2 * i + 1];
  return t[0];
}

// One warp per lattice row: finishes the x-tree over the nseg segment partials of that row.
__global__ void __launch_bounds__(256) row_reduce_kernel(const __grid_constant__ ReduceArgs p) {
  const int b = blockIdx.y;
  const int row = blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (row >= p.Ny) return;
  int P = 32;
  while (P < p.nseg) P <<= 1;
  const int m = P / 32;
  const long long base = ((long long)b * p.Ny + row) * p.nseg;
  const double* src[3] = {p.part_e + base, p.part_q + base, p.part_ke + base};
#pragma unroll
  for (int qn = 0; qn < 3; ++qn) {
    double v = chunk_tree(src[qn], (long long)lane * m, p.nseg, m);
    v = warp_tree(v);
    if (lane == 0) p.rows[((long long)b * 3 + qn) * p.Ny + row] = v;
  }
}

// One CTA per lattice: y-tree over the row sums, E/Q/KE, arrest decision (eq. 4).
__global__ void __launch_bounds__(1024) finalize_kernel(const __grid_constant__ ReduceArgs p) {
  __shared__ double sh[3][32];
  const int b = blockIdx.x;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  int P = 1024;
  while (P < p.Ny) P <<= 1;
  const int m = P / 1024;
  double tot[3];
#pragma unroll
  for (int qn = 0; qn < 3; ++qn) {
    const double* src = p.rows + ((long long)b * 3 + qn) * p.Ny;
    double v = chunk_tree(src, (long long)t * m, p.Ny, m);
    v = warp_tree(v);
    if (lane == 0) sh[qn][wid] = v;
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int qn = 0; qn < 3; ++qn) tot[qn] = warp_tree(sh[qn][lane]);
    if (lane == 0) {
      LatticeState& st = p.state[b];
      const double E = p.h2 * tot[0], Q = p.h2 * tot[1], KE = p.h2 * tot[2];
      st.step += p.advance;
      const bool arrest = E > st.E_prev;  // strict; NaN compares false
      if (!isfinite(E)) st.nonfinite = 1;
      st.v_is_zero = arrest ? 1 : 0;
      if (arrest) {
        if (st.n_arrests < p.log_cap) p.log[(long long)b * p.log_cap + st.n_arrests] = st.step;
        st.n_arrests += 1;
      }
      st.E = E;
      st.Q = Q;
      st.KE = KE;
      st.E_prev = E;
    }
  }
}

// ------------------------------------------------------------------ set / get helpers
template <typename real>
__global__ void copy_interior_kernel(real* dst, const real* src, int Nx, int Ny, long long planes) {
  const long long n = planes * Nx * Ny;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const int x = int(i % Nx), y = int((i / Nx) % Ny);
    const bool inter = x >= HALO && x < Nx - HALO && y >= HALO && y < Ny - HALO;
    dst[i] = inter ? src[i] : real(0);
  }
}

// velocity read-out: exactly 0 on lattices whose last step was arrested
template <typename real>
__global__ void export_velocity_kernel(real* dst, const real* src, const LatticeState* state,
                                       long long per_lattice, int batch) {
  const long long n = per_lattice * batch;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const int b = int(i / per_lattice);
    dst[i] = state[b].v_is_zero ? real(0) : src[i];
  }
}

__global__ void init_state_kernel(LatticeState* state, int batch) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= batch) return;
  LatticeState s;
  s.E = 0.0; s.Q = 0.0; s.KE = 0.0;
  s.E_prev = __longlong_as_double(0x7ff0000000000000LL);  // +inf: step 0 cannot arrest
  s.n_arrests = 0; s.step = 0; s.v_is_zero = 0; s.nonfinite = 0;
  state[b] = s;
}

}  // namespace ss
