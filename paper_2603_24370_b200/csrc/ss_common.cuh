// Shared device-side definitions of libss.so (CUDA, sm_100a).  No code here is shared with
// oracle/: the oracle is an independent plain-C statement of the same mathematics.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ss {

// kernel families: kCMG = chiral magnet with a general DMI table, kBS = baby Skyrme
constexpr int kCM = 0, kAH = 1, kCMG = 2, kBS = 3;
constexpr int HALO = 2;  // PAPER.md:102 "fourth-order ... stencils and halo width two"

// Row segment of the canonical reduction tree (DESIGN R10): per-row partial sums are stored
// for aligned segments of SEG consecutive x.  All stencil kernels use tiles SEG wide.
constexpr int SEG = 64;

// Per-lattice scalars kept on the device (PAPER.md:158 reductions; eq. 4 arrest state).
struct LatticeState {
  double E, Q, KE, E_prev;
  long long n_arrests, step;
  int v_is_zero, nonfinite;
};

struct ReduceArgs {
  const double* part_e;  // [batch][Ny][nseg]
  const double* part_q;
  const double* part_ke;
  double* rows;          // [batch][3][Ny] row sums
  LatticeState* state;
  long long* log;        // [batch][log_cap]
  long long log_cap;
  int Ny, nseg, advance;
  double h2;             // h*h
  int row0, row1;        // row_reduce: this launch finishes rows [row0, row1)
};

// Aligned pairwise tree over the 32 lanes of a warp (lane l holds element l):
// xor-shuffles realise t[m] = t[2m] + t[2m+1] level by level because IEEE addition commutes.
__device__ __forceinline__ double warp_tree(double v) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Two horizontally adjacent fp32 sites computed side by side with the packed fp32 instructions of
// sm_100 (FFMA2 / FADD2 / FMUL2): the fp32 build of the flow kernels is issue-bound, and one
// thread owning the pair (x, x+1) halves both the arithmetic and the shared-memory instructions.
struct f2 {
  float2 v;
  f2() = default;
  __device__ __forceinline__ f2(float a) : v(make_float2(a, a)) {}
  __device__ __forceinline__ f2(double a) : v(make_float2(float(a), float(a))) {}
  __device__ __forceinline__ f2(int a) : v(make_float2(float(a), float(a))) {}
  __device__ __forceinline__ f2(float a, float b) : v(make_float2(a, b)) {}
  __device__ __forceinline__ explicit f2(float2 t) : v(t) {}
};
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return f2(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { return f2(__fmul2_rn(a.v, b.v)); }
__device__ __forceinline__ f2 operator-(f2 a) { return f2(make_float2(-a.v.x, -a.v.y)); }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { return a + (-b); }
__device__ __forceinline__ f2 operator*(float a, f2 b) { return f2(a) * b; }
__device__ __forceinline__ f2 operator*(f2 a, float b) { return a * f2(b); }
__device__ __forceinline__ f2 operator+(f2 a, float b) { return a + f2(b); }
__device__ __forceinline__ f2 operator+(float a, f2 b) { return f2(a) + b; }
__device__ __forceinline__ f2 operator-(f2 a, float b) { return a - f2(b); }
__device__ __forceinline__ f2 operator-(float a, f2 b) { return f2(a) - b; }
__device__ __forceinline__ f2& operator+=(f2& a, f2 b) { a = a + b; return a; }
__device__ __forceinline__ f2& operator-=(f2& a, f2 b) { a = a - b; return a; }
__device__ __forceinline__ f2& operator*=(f2& a, f2 b) { a = a * b; return a; }
// fused multiply-add written as a * b + c contracts to FFMA2 only through the intrinsic
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return f2(__ffma2_rn(a.v, b.v, c.v)); }

template <typename real> __device__ __forceinline__ real rsqrt_(real x);
template <> __device__ __forceinline__ f2 rsqrt_<f2>(f2 x) { return f2(rsqrtf(x.v.x), rsqrtf(x.v.y)); }
template <> __device__ __forceinline__ double rsqrt_<double>(double x) { return rsqrt(x); }
template <> __device__ __forceinline__ float rsqrt_<float>(float x) { return rsqrtf(x); }

}  // namespace ss
