// Headless visualisation kernels ("extrema used for visualization ... parallel
// GPU reductions"; "visualization kernels then write image data directly into this buffer ...
// energy density, order-parameter magnitude, magnetic flux density").  The CUDA half only: the
// image goes to a plain device buffer, there is no GL interop on this box (DESIGN R17).
//
//   observable_kernel  per-site observable (fp64) of one lattice -> per-block min / max over the
//                      finite interior values; flags a non-finite one
//   minmax_kernel      extrema over the block partials (min / max are order independent: exact)
//   colormap_kernel    the observable again, t = (v - min) / (max - min) -> RGBA8 through a 5-stop
//                      piecewise-linear map (own definition, DESIGN R17); halo sites (by position)
//                      are transparent black, non-finite values opaque magenta
#pragma once
#include "ss_flow.cuh"

namespace ss {

constexpr int OBS_ENERGY = 0, OBS_CHARGE = 1, OBS_ORDER = 2;

template <typename real>
struct RenderArgs {
  const real* phi;      // [C][Ny][Nx] of the lattice
  double* part;         // [nblocks][2] block min, max
  double* minmax;       // [2]
  int* nonfinite;       // set when an interior value is NaN / Inf (zeroed by the host first)
  unsigned int* rgba;   // [Ny][Nx]
  int Nx, Ny, obs, nblocks;
  real B;
};

// observable of interior site (gx, gy) in fp64; both passes (extrema, colour map) evaluate it with
// this one routine on the same inputs, so they see identical values and no scratch plane is needed
template <int THEORY, typename real>
__device__ __forceinline__ double observable_at(const FlowArgs<real>& p, const RenderArgs<real>& r,
                                                int gx, int gy) {
  using Th = typename TheoryOf<THEORY, real>::type;
  const long long plane = (long long)r.Nx * r.Ny;
  auto T = [&](int c, int dy, int dx) -> real {
    return r.phi[c * plane + (long long)(gy + dy) * r.Nx + gx + dx];
  };
  if (r.obs == OBS_ORDER)
    return THEORY == kAH ? sqrt(double(T(0, 0, 0)) * double(T(0, 0, 0)) +
                                double(T(1, 0, 0)) * double(T(1, 0, 0)))
                         : double(T(2, 0, 0));
  real e, q;
  Th::densities(T, p, r.B, EdgeW(gx, gy, r.Nx, r.Ny), e, q);
  return r.obs == OBS_ENERGY ? double(e) : double(q);
}

__device__ __forceinline__ bool interior_site(int gx, int gy, int Nx, int Ny) {
  return gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO;
}

template <int THEORY, typename real>
__global__ void __launch_bounds__(256) observable_kernel(const __grid_constant__ FlowArgs<real> p,
                                                         const __grid_constant__ RenderArgs<real> r) {
  __shared__ double smn[8], smx[8];
  const int Nx = r.Nx, Ny = r.Ny;
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  double mn = inf, mx = -inf;  // halo sites and non-finite values do not enter the extrema
  if (i < (long long)Nx * Ny) {
    const int gx = int(i % Nx), gy = int(i / Nx);
    if (interior_site(gx, gy, Nx, Ny)) {
      const double v = observable_at<THEORY, real>(p, r, gx, gy);
      if (isfinite(v)) mn = mx = v;
      else atomicOr(r.nonfinite, 1);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
    mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  }
  if ((threadIdx.x & 31) == 0) { smn[threadIdx.x >> 5] = mn; smx[threadIdx.x >> 5] = mx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < 8; ++k) { mn = fmin(mn, smn[k]); mx = fmax(mx, smx[k]); }
    r.part[2 * blockIdx.x] = mn;
    r.part[2 * blockIdx.x + 1] = mx;
  }
}

template <typename real>
__global__ void __launch_bounds__(1024) minmax_kernel(const __grid_constant__ RenderArgs<real> r) {
  __shared__ double smn[32], smx[32];
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  double mn = inf, mx = -inf;
  for (int k = threadIdx.x; k < r.nblocks; k += 1024) {
    mn = fmin(mn, r.part[2 * k]);
    mx = fmax(mx, r.part[2 * k + 1]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
    mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  }
  if ((threadIdx.x & 31) == 0) { smn[threadIdx.x >> 5] = mn; smx[threadIdx.x >> 5] = mx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < 32; ++k) { mn = fmin(mn, smn[k]); mx = fmax(mx, smx[k]); }
    r.minmax[0] = mn;
    r.minmax[1] = mx;
  }
}

// 5 stops at t = 0, 1/4, 1/2, 3/4, 1 (dark blue, azure, white, orange, dark red); every operation
// is a single IEEE fp64 operation in a fixed order (no contraction) so that the byte decisions are
// reproducible on a CPU.  Halo sites (by position): transparent black; a non-finite interior
// value: opaque magenta.
template <int THEORY, typename real>
__global__ void __launch_bounds__(256) colormap_kernel(const __grid_constant__ FlowArgs<real> p,
                                                       const __grid_constant__ RenderArgs<real> r) {
  const double stops[5][3] = {{0, 0, 128}, {0, 128, 255}, {255, 255, 255}, {255, 128, 0}, {128, 0, 0}};
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i >= (long long)r.Nx * r.Ny) return;
  const int gx = int(i % r.Nx), gy = int(i / r.Nx);
  unsigned int out = 0u;
  if (interior_site(gx, gy, r.Nx, r.Ny)) {
    const double v = observable_at<THEORY, real>(p, r, gx, gy);
    const double mn = r.minmax[0], mx = r.minmax[1];
    if (!isfinite(v)) {
      out = 0xffff00ffu;
    } else {
      const double span = __dsub_rn(mx, mn);
      const double t = span > 0.0 ? __ddiv_rn(__dsub_rn(v, mn), span) : 0.5;
      const double t4 = __dmul_rn(t, 4.0);
      int seg = int(t4);
      seg = seg > 3 ? 3 : seg;
      const double u = __dsub_rn(t4, double(seg));
      unsigned int ch[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const double c0 = stops[seg][k], c1 = stops[seg + 1][k];
        const double x = __dadd_rn(__dadd_rn(c0, __dmul_rn(__dsub_rn(c1, c0), u)), 0.5);
        ch[k] = (unsigned int)int(floor(x));
      }
      out = ch[0] | (ch[1] << 8) | (ch[2] << 16) | (255u << 24);
    }
  }
  r.rgba[i] = out;
}

}  // namespace ss
