// Demagnetisation of the chiral magnet (eq. (5) last term, :199-205 eq. (6);
// DESIGN R19): the magnetostatic potential psi, (Lx + Ly) psi = D_x n1 + D_y n2
// on the interior with psi = 0 on the halo, is solved on the device by geometric multigrid
// V-cycles, and enters the one-gradient-per-step (velocity Verlet, DESIGN R15) flow step:
//
//   demag_drift_kernel   w = vh + dt/2 a, phi' = R(phi + dt w)                    (pointwise)
//   demag_rho_kernel     rho = D_x n1' + D_y n2'                                  (eq. 1)
//   mg_* kernels         n V-cycles V(2,2) on psi, warm-started from the previous step:
//                        damped-Jacobi smoothing of the 4th-order operator (omega = 10/13, the
//                        optimum for its symbol: smoothing factor 0.64), cell-centred
//                        coarsening by 2 (4-point averaging down, bilinear up; an odd size drops
//                        its last cell: n_c = floor(n/2)), the same eq. (2) operator with
//                        h_l = 2^l h on every level, each coarse level closed by wall images at
//                        its exact distance from the physical wall, coarsest level (<= 8 x 8)
//                        relaxed to convergence by one CTA
//   demag_kick_kernel    a' = -Pi(G(phi') + g (D_x psi, D_y psi, 0)), e_i + g x bond density of
//                        psi, q_i, v' = Pi(w + dt/2 a'), KE, row-segment partial sums
// and the RK4 step with one solve per stage field: for stages 2, 3, 4
// demag_stage_kernel (S = R(phi + alpha vh + beta a_prev)) -> demag_rho -> V-cycles -> demag_kick
// (acceleration only), then demag_combine_kernel (phi', v', KE) and rho -> V-cycles -> kick (a1,
// e, q) on phi'.  psi is warm-started from the previous solve throughout.
//
// Roofline (stated before the kernels were written): HBM, but not 10 C R.  Per
// interior site and step in fp64: drift 5 C R = 120 B, rho 3 R = 24 B, kick 13 R = 104 B, and
// per V-cycle 4 sweeps x 3 R + residual/restriction 2.25 R + prolongation 2.25 R = 16.5 R on the
// finest level, x 4/3 for the coarser ones = 22 R = 176 B:  248 + 176 n_cycles bytes.
#pragma once
#include "ss_flow.cuh"

namespace ss {

constexpr int MGX = 32, MGY = 8;          // thread block of the multigrid kernels
constexpr int MG_COARSE_MAX = 8;          // coarsen until both sizes are <= 8 (or one reaches 2)
constexpr int MG_COARSE_SWEEPS = 40;       // measured: 40 sweeps keep the V-cycle at 0.27, 20 do not
constexpr double MG_OMEGA = 10.0 / 13.0;  // 1 - 28 w/60 = -(1 - 128 w/60)

// A level holds nx x ny unknowns inside a zero halo of width 2: arrays [batch][ny+4][nx+4].
// arguments of every multigrid kernel (which members are used depends on the kernel)
struct MgArgs {
  double* out;        // smooth: new iterate; restrict: coarse rhs; prolong: fine psi; coarse: psi
  double* out2;       // restrict: coarse psi (zeroed)
  const double* in;   // smooth: old iterate; restrict: fine psi; prolong: coarse psi
  const double* rhs;  // smooth, restrict, coarse
  int nx, ny;         // fine (or only) level
  int cnx, cny;       // coarse level
  double c;           // 1 / (12 h_l^2) of the level the operator is applied on
  int walls;          // 0 on level 0 (plain zero halo); 1: the level's halo holds wall images
  double bw[8];       // image factors of the output level: (beta1, beta2) for the left, right,
                      // bottom and top wall (see mg_store)
};

// Wall treatment.  Level 0 is the lattice: psi = 0 on its two halo layers (the wall sits on the
// first halo node, one spacing from the first unknown).  On a cell-centred coarse level l >= 1 the
// first / last unknown lies d spacings OF THAT LEVEL from the same physical wall -- d = 1/2 +
// 1/2^(l+1) on the left and bottom, and on the right and top whatever the dropped cells of the
// odd sizes above leave (1.0 ... 1.25 right after a drop).  Its two halo layers hold the values of
// the straight line through the wall and the wall-adjacent unknown: psi(-k) = beta_k psi(0),
// beta_k = (d - k)/d.  Whoever writes a wall-adjacent cell of such a level also writes its
// images (corners: the product), so every kernel reads plain neighbours.
__device__ __forceinline__ void mg_store(double* q, int i, int j, int nx, int ny, int pitch,
                                         double v, int walls, const double* bw) {
  q[0] = v;
  if (!walls) return;
  const bool L = i == 0, R = i == nx - 1, B = j == 0, T = j == ny - 1;
  if (!(L || R || B || T)) return;
#pragma unroll
  for (int k = 1; k <= 2; ++k) {
    if (L) q[-k] = bw[k - 1] * v;
    if (R) q[k] = bw[2 + k - 1] * v;
    if (B) q[-k * pitch] = bw[4 + k - 1] * v;
    if (T) q[k * pitch] = bw[6 + k - 1] * v;
  }
  // corners, read only by the bilinear prolongation from this level (nearest image only)
  if (L && B) q[-pitch - 1] = bw[0] * bw[4] * v;
  if (R && B) q[-pitch + 1] = bw[2] * bw[4] * v;
  if (L && T) q[pitch - 1] = bw[0] * bw[6] * v;
  if (R && T) q[pitch + 1] = bw[2] * bw[6] * v;
}

__device__ __forceinline__ double mg_lap(const double* q, int pitch, double c) {
  // (Lx + Ly) psi at *q  (eq. 2 in both directions)
  return c * ((16.0 * ((q[1] + q[-1]) + (q[pitch] + q[-pitch])) -
               ((q[2] + q[-2]) + (q[2 * pitch] + q[-2 * pitch]))) -
              60.0 * q[0]);
}

// out = in + omega (rhs - L in) / diag(L),  diag(L) = -60 c
__global__ void __launch_bounds__(MGX* MGY) mg_smooth_kernel(const __grid_constant__ MgArgs m) {
  const int nx = m.nx, ny = m.ny;
  const double c = m.c;
  const double* in = m.in;
  const double* rhs = m.rhs;
  double* out = m.out;
  const int i = blockIdx.x * MGX + threadIdx.x, j = blockIdx.y * MGY + threadIdx.y;
  if (i >= nx || j >= ny) return;
  const int pitch = nx + 4;
  const long long o = ((long long)blockIdx.z * (ny + 4) + j + 2) * pitch + i + 2;
  const double r = rhs[o] - mg_lap(in + o, pitch, c);
  mg_store(out + o, i, j, nx, ny, pitch, in[o] - (MG_OMEGA / (60.0 * c)) * r, m.walls, m.bw);
}

// coarse rhs = average of the residuals of the four fine children; coarse psi = 0
__global__ void __launch_bounds__(MGX* MGY) mg_restrict_kernel(const __grid_constant__ MgArgs m) {
  const int nx = m.nx, ny = m.ny, cnx = m.cnx, cny = m.cny;
  const double c = m.c;
  const double* psi = m.in;
  const double* rhs = m.rhs;
  double* crhs = m.out;
  double* cpsi = m.out2;
  const int I = blockIdx.x * MGX + threadIdx.x, J = blockIdx.y * MGY + threadIdx.y;
  if (I >= cnx || J >= cny) return;
  const int pitch = nx + 4;
  const long long base = (long long)blockIdx.z * (ny + 4) * pitch;
  double s = 0.0;
#pragma unroll
  for (int dj = 0; dj < 2; ++dj)
#pragma unroll
    for (int di = 0; di < 2; ++di) {  // cnx = nx / 2, cny = ny / 2: all four children exist
      const long long o = base + (long long)(2 * J + dj + 2) * pitch + 2 * I + di + 2;
      s += rhs[o] - mg_lap(psi + o, pitch, c);
    }
  const long long co = ((long long)blockIdx.z * (cny + 4) + J + 2) * (cnx + 4) + I + 2;
  crhs[co] = 0.25 * s;
  mg_store(cpsi + co, I, J, cnx, cny, cnx + 4, 0.0, 1, m.bw);  // zero the stale images too
}

// psi_fine += bilinear (cell-centred) interpolation of the coarse correction (the last cell of an
// odd size has no parent: it interpolates between its neighbour's parent and the zero wall)
__global__ void __launch_bounds__(MGX* MGY) mg_prolong_kernel(const __grid_constant__ MgArgs m) {
  const int nx = m.nx, ny = m.ny, cnx = m.cnx, cny = m.cny;
  double* psi = m.out;
  const double* cpsi = m.in;
  const int i = blockIdx.x * MGX + threadIdx.x, j = blockIdx.y * MGY + threadIdx.y;
  if (i >= nx || j >= ny) return;
  const int cp = cnx + 4;
  const int I = i >> 1, J = j >> 1, sx = (i & 1) ? 1 : -1, sy = (j & 1) ? 1 : -1;
  const double* q = cpsi + ((long long)blockIdx.z * (cny + 4) + J + 2) * cp + I + 2;
  const double v = (9.0 * q[0] + 3.0 * (q[sx] + q[sy * cp]) + q[sy * cp + sx]) * (1.0 / 16.0);
  psi[((long long)blockIdx.z * (ny + 4) + j + 2) * (nx + 4) + i + 2] += v;
}

// coarsest level: one CTA per lattice, damped Jacobi to convergence in shared memory
__global__ void __launch_bounds__(1024) mg_coarse_kernel(const __grid_constant__ MgArgs m) {
  const int nx = m.nx, ny = m.ny;
  const double c = m.c;
  double* psi = m.out;
  const double* rhs = m.rhs;
  extern __shared__ double sh[];
  const int pitch = nx + 4, n = (nx + 4) * (ny + 4);
  double *a = sh, *b2 = sh + n, *r = sh + 2 * n;
  const long long base = (long long)blockIdx.x * n;
  for (int k = threadIdx.x; k < n; k += blockDim.x) {
    a[k] = psi[base + k];  // 0 below level 0 (zeroed by the restriction); the warm start on level 0
    b2[k] = 0.0;
    r[k] = rhs[base + k];
  }
  __syncthreads();
  for (int it = 0; it < MG_COARSE_SWEEPS; ++it) {
    for (int k = threadIdx.x; k < nx * ny; k += blockDim.x) {
      const int o = (k / nx + 2) * pitch + k % nx + 2;
      mg_store(b2 + o, k % nx, k / nx, nx, ny, pitch,
               a[o] - (MG_OMEGA / (60.0 * c)) * (r[o] - mg_lap(a + o, pitch, c)), m.walls, m.bw);
    }
    __syncthreads();
    double* t = a; a = b2; b2 = t;
  }
  for (int k = threadIdx.x; k < nx * ny; k += blockDim.x) {
    const int o = (k / nx + 2) * pitch + k % nx + 2;
    mg_store(psi + base + o, k % nx, k / nx, nx, ny, pitch, a[o], m.walls, m.bw);
  }
}

// ------------------------------------------------------------------ the flow step around it
struct DemagArgs {
  const double* phi;   // [batch][3][Ny][Nx] field the kernel reads (drift: phi^n; rho, kick: phi')
  const double* vel;   // drift: v^n; kick: w (half-kicked velocity)
  const double* acc;   // drift: a(phi^n)
  double* phi_out;     // drift: phi'
  double* vel_out;     // drift: w; kick: v'
  double* acc_out;     // kick: a(phi')
  double* rho;         // [batch][Ny][Nx]
  const double* psi;   // [batch][Ny][Nx], halo 0
  double* part_e;      // [batch][Ny][nseg]
  double* part_q;
  double* part_ke;
  const LatticeState* state;
  const double* Bb;
  int advance;         // kick: 1 = second half kick + KE; 0 = evaluation (a, e, q); 2 = a only
  double g;            // mu0 Ms^2
  // RK4 with demagnetisation (one Poisson solve per stage field)
  const double* a1;    // combine: the four stage accelerations
  const double* a2;
  const double* a3;
  const double* a4;
  double alpha, beta;  // stage: S = R(phi + alpha vh + beta acc)
  int use_acc;         // stage: 0 for stage 2 (no acceleration term)
};
struct DemagStepArgs {
  FlowArgs<double> p;  // per-site constants (tensor maps unused)
  DemagArgs d;
};

__global__ void __launch_bounds__(256) demag_drift_kernel(const __grid_constant__ DemagStepArgs A) {
  const FlowArgs<double>& p = A.p;
  const DemagArgs& d = A.d;
  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z;
  const bool vz = d.state[b].v_is_zero != 0;
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i >= p.plane) return;
  const int x = int(i % Nx), y = int(i / Nx);
  if (x < HALO || x >= Nx - HALO || y < HALO || y >= Ny - HALO) return;
  const long long lat = (long long)b * 3 * p.plane;
  double m[3], w[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const long long o = lat + c * p.plane + i;
    const double vh = vz ? 0.0 : d.vel[o];
    w[c] = vh + p.hdt * d.acc[o];
    m[c] = d.phi[o] + p.dt * w[c];
  }
  CM<double>::project_field(m);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    d.phi_out[lat + c * p.plane + i] = m[c];
    d.vel_out[lat + c * p.plane + i] = w[c];
  }
}

// RK4 stage field S = R(phi + alpha vh [+ beta a_prev]) on the interior (PAPER.md:123, :129+154;
// the same expressions as the oracle's stage_field), written where phi' will go later
__global__ void __launch_bounds__(256) demag_stage_kernel(const __grid_constant__ DemagStepArgs A) {
  const FlowArgs<double>& p = A.p;
  const DemagArgs& d = A.d;
  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z;
  const bool vz = d.state[b].v_is_zero != 0;
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i >= p.plane) return;
  const int x = int(i % Nx), y = int(i / Nx);
  if (x < HALO || x >= Nx - HALO || y < HALO || y >= Ny - HALO) return;
  const long long lat = (long long)b * 3 * p.plane;
  double m[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const long long o = lat + c * p.plane + i;
    const double vh = vz ? 0.0 : d.vel[o];
    m[c] = d.phi[o] + d.alpha * vh;
    if (d.use_acc) m[c] = m[c] + d.beta * d.acc[o];
  }
  CM<double>::project_field(m);
#pragma unroll
  for (int c = 0; c < 3; ++c) d.phi_out[lat + c * p.plane + i] = m[c];
}

__global__ void __launch_bounds__(256) demag_rho_kernel(const __grid_constant__ DemagStepArgs A) {
  const FlowArgs<double>& p = A.p;
  const DemagArgs& d = A.d;
  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z;
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i >= p.plane) return;
  const int x = int(i % Nx), y = int(i / Nx);
  if (x < HALO || x >= Nx - HALO || y < HALO || y >= Ny - HALO) return;
  const double* n1 = d.phi + (long long)b * 3 * p.plane + i;
  const double* n2 = n1 + p.plane;
  d.rho[(long long)b * p.plane + i] =
      p.i12h * (d1n<double>(n1[-2], n1[-1], n1[1], n1[2]) +
                d1n<double>(n2[-2 * Nx], n2[-Nx], n2[Nx], n2[2 * Nx]));
}

constexpr int DTX = SEG, DTY = 16, DBX = 64, DBY = 4;

template <int THEORY>
__global__ void __launch_bounds__(DBX* DBY) demag_kick_kernel(const __grid_constant__ DemagStepArgs A) {
  const FlowArgs<double>& p = A.p;
  const DemagArgs& d = A.d;
  using Th = typename TheoryOf<THEORY, double>::type;
  __shared__ double sm[4][DTY + 2 * HALO][DTX + 2 * HALO];  // phi' (3) and psi
  __shared__ double red[3][DTY][DBX / 32];
  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z, x0 = blockIdx.x * DTX, y0 = blockIdx.y * DTY;
  const long long lat = (long long)b * 3 * p.plane;
  const int tid = threadIdx.y * DBX + threadIdx.x;
  for (int idx = tid; idx < (DTY + 2 * HALO) * (DTX + 2 * HALO); idx += DBX * DBY) {
    const int ly = idx / (DTX + 2 * HALO), lx = idx - ly * (DTX + 2 * HALO);
    const int gx = x0 - HALO + lx, gy = y0 - HALO + ly;
    const bool in = gx >= 0 && gx < Nx && gy >= 0 && gy < Ny;
    const long long o = (long long)gy * Nx + gx;
#pragma unroll
    for (int c = 0; c < 3; ++c) sm[c][ly][lx] = in ? d.phi[lat + c * p.plane + o] : 0.0;
    sm[3][ly][lx] = in ? d.psi[(long long)b * p.plane + o] : 0.0;
  }
  __syncthreads();
  const double Bz = d.Bb[b];
  const int gx = x0 + threadIdx.x;
  const int warp_in_row = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll 1
  for (int r = 0; r < DTY / DBY; ++r) {
    const int ly = r * DBY + threadIdx.y, gy = y0 + ly;
    const bool active = gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    if (active) {
      const int cx = threadIdx.x + HALO, cy = ly + HALO;
      auto T = [&](int c, int dy, int dx) -> double { return sm[c][cy + dy][cx + dx]; };
      const double n[3] = {T(0, 0, 0), T(1, 0, 0), T(2, 0, 0)};
      double G[3];
      Th::gradient(T, p, Bz, G);
      G[0] += d.g * (p.i12h * Dxn<double>(T, 3));
      G[1] += d.g * (p.i12h * Dyn<double>(T, 3));
      const double gn = (G[0] * n[0] + G[1] * n[1]) + G[2] * n[2];
      const double a[3] = {gn * n[0] - G[0], gn * n[1] - G[1], gn * n[2] - G[2]};
      double e = 0.0, q = 0.0;
      const EdgeW w(gx, gy, Nx, Ny);
      if (d.advance != 2) Th::densities(T, p, Bz, w, e, q);
      if (d.advance != 2) {  // + g x bond density of psi (site form, halo weights R3)
        const int ks[4] = {1, -1, 2, -2};
        double sA = 0.0, sB = 0.0;
#pragma unroll
        for (int s = 0; s < 4; ++s) {
          const double ax = T(3, 0, 0) - T(3, 0, ks[s]), ay = T(3, 0, 0) - T(3, ks[s], 0);
          const double t = double(w.wx(s)) * (ax * ax) + double(w.wy(s)) * (ay * ay);
          if (s < 2) sA += t; else sB += t;
        }
        e += d.g * (p.jA * sA + p.jB * sB);
      }
      s0 = e;
      s1 = q;
      const long long o = (long long)gy * Nx + gx;
      if (d.advance == 1) {
        double u[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) u[c] = d.vel[lat + c * p.plane + o] + p.hdt * a[c];
        Th::project_velocity(u, n);
        double v2 = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          d.vel_out[lat + c * p.plane + o] = u[c];
          v2 += u[c] * u[c];
        }
        s2 = 0.5 * v2;
      }
#pragma unroll
      for (int c = 0; c < 3; ++c) d.acc_out[lat + c * p.plane + o] = a[c];
    }
    s0 = warp_tree(s0);
    s1 = warp_tree(s1);
    s2 = warp_tree(s2);
    if (lane == 0) {
      red[0][ly][warp_in_row] = s0;
      red[1][ly][warp_in_row] = s1;
      red[2][ly][warp_in_row] = s2;
    }
  }
  __syncthreads();
  if (d.advance != 2 && tid < DTY && y0 + tid < Ny) {
    const long long po = ((long long)b * Ny + (y0 + tid)) * p.nseg + blockIdx.x;
    d.part_e[po] = red[0][tid][0] + red[0][tid][1];
    d.part_q[po] = red[1][tid][0] + red[1][tid][1];
    if (d.advance == 1) d.part_ke[po] = red[2][tid][0] + red[2][tid][1];
  }
}

// RK4 combine (the oracle's expressions): phi' = R((phi + dt vh) + dt^2/6 ((a1 + a2)
// + a3)), u = vh + dt/6 ((a1 + 2 a2) + (2 a3 + a4)), v' = u - (u.phi') phi', KE partial sums
__global__ void __launch_bounds__(DBX* DBY) demag_combine_kernel(const __grid_constant__ DemagStepArgs A) {
  const FlowArgs<double>& p = A.p;
  const DemagArgs& d = A.d;
  __shared__ double red[DTY][DBX / 32];
  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z, x0 = blockIdx.x * DTX, y0 = blockIdx.y * DTY;
  const long long lat = (long long)b * 3 * p.plane;
  const int tid = threadIdx.y * DBX + threadIdx.x;
  const bool vz = d.state[b].v_is_zero != 0;
  const int gx = x0 + threadIdx.x;
  const int warp_in_row = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll 2
  for (int r = 0; r < DTY / DBY; ++r) {
    const int ly = r * DBY + threadIdx.y, gy = y0 + ly;
    double s0 = 0.0;
    if (gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO) {
      const long long o = (long long)gy * Nx + gx;
      double f[3], u[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const long long oc = lat + c * p.plane + o;
        const double vh = vz ? 0.0 : d.vel[oc];
        const double A1 = d.a1[oc], A2 = d.a2[oc], A3 = d.a3[oc], A4 = d.a4[oc];
        f[c] = (d.phi[oc] + p.dt * vh) + p.sdt2 * ((A1 + A2) + A3);
        u[c] = vh + p.sdt * ((A1 + 2.0 * A2) + (2.0 * A3 + A4));
      }
      CM<double>::project_field(f);
      CM<double>::project_velocity(u, f);
      double v2 = 0.0;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        d.phi_out[lat + c * p.plane + o] = f[c];
        d.vel_out[lat + c * p.plane + o] = u[c];
        v2 += u[c] * u[c];
      }
      s0 = 0.5 * v2;
    }
    s0 = warp_tree(s0);
    if (lane == 0) red[ly][warp_in_row] = s0;
  }
  __syncthreads();
  if (tid < DTY && y0 + tid < Ny)
    d.part_ke[((long long)b * Ny + (y0 + tid)) * p.nseg + blockIdx.x] = red[tid][0] + red[tid][1];
}

}  // namespace ss
