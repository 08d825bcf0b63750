// Small kernels of the flow step: the two reduction kernels that finish the canonical tree
// (DESIGN R10) and take the arrest decision (eq. 4) on the device, and the helpers of
// ss_set_fields / ss_get_fields.  The stencil work is in ss_flow.cuh.
#pragma once
#include "ss_theory.cuh"

namespace ss {

// In-thread aligned pairwise tree over m (power of two, <= 32) consecutive values: all loads are
// issued first, the tree runs in registers (one instance per m).
template <int M>
__device__ __forceinline__ double chunk_tree_m(const double* src, long long first, long long n) {
  double t[M];
#pragma unroll
  for (int i = 0; i < M; ++i) t[i] = (first + i < n) ? src[first + i] : 0.0;
#pragma unroll
  for (int s = M; s > 1; s >>= 1)
#pragma unroll
    for (int i = 0; i < s / 2; ++i) t[i] = t[2 * i] + t[2 * i + 1];
  return t[0];
}
__device__ __forceinline__ double chunk_tree(const double* src, long long first, long long n, int m) {
  switch (m) {
    case 1: return chunk_tree_m<1>(src, first, n);
    case 2: return chunk_tree_m<2>(src, first, n);
    case 4: return chunk_tree_m<4>(src, first, n);
    case 8: return chunk_tree_m<8>(src, first, n);
    case 16: return chunk_tree_m<16>(src, first, n);
    default: return chunk_tree_m<32>(src, first, n);
  }
}

// One warp per lattice row: finishes the x-tree over the nseg segment partials of that row.
__global__ void __launch_bounds__(256) row_reduce_kernel(const __grid_constant__ ReduceArgs p) {
  const int b = blockIdx.y;
  const int row = p.row0 + blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (row >= p.row1) return;
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

// the second ping-pong buffers: frozen halo of phi copied from the first, halo of v zero (a step
// writes their interior before anything reads it); 4 (Nx + Ny - 4) sites per plane
template <typename real>
__global__ void init_halo_kernel(real* phi1, real* vel1, const real* phi0, int Nx, int Ny,
                                 long long planes) {
  const long long ring = 2LL * HALO * Nx + 2LL * HALO * (Ny - 2 * HALO);
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < planes * ring;
       i += (long long)gridDim.x * blockDim.x) {
    const long long pl = i / ring;
    long long r = i % ring;
    int x, y;
    if (r < 2LL * HALO * Nx) {  // rows 0, 1, Ny-2, Ny-1
      const int k = int(r / Nx);
      y = k < HALO ? k : Ny - 2 * HALO + k;
      x = int(r % Nx);
    } else {                    // columns 0, 1, Nx-2, Nx-1 of the other rows
      r -= 2LL * HALO * Nx;
      const int k = int(r % (2 * HALO));
      y = HALO + int(r / (2 * HALO));
      x = k < HALO ? k : Nx - 2 * HALO + k;
    }
    const long long o = (pl * Ny + y) * Nx + x;
    phi1[o] = phi0[o];
    vel1[o] = real(0);
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
