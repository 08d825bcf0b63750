// Two-kernel flow step: y-marching strips, TMA-staged chunks, smem rings.
//
//   flow_kernel<THEORY, real, KX>  "X": reads phi, v            -> writes a1, a2, E/Q partials
//       a1 = -Pi G(phi), e_i, q_i          (PAPER.md:104-109 stencils, :158 reductions)
//       a2 = -Pi G(phi2), phi2 = R(phi + dt/2 v)   (RK4 stage 2 assuming "not arrested";
//                                           an arrested step uses a2 := a1, DESIGN R11)
//   flow_kernel<THEORY, real, KY>  "Y": reads phi, v, a1, a2    -> writes phi', v', KE partials
//       phi3 = R((phi + dt/2 vh) + dt^2/4 a1), a3 = -Pi G(phi3)
//       phi4 = R((phi + dt vh) + dt^2/2 a2),   a4 = -Pi G(phi4)
//       RK4 combine + projections (PAPER.md:123, :129+154), vh = arrested ? 0 : v (eq. 4)
//
// A CTA owns a strip of FW = 64 columns and a segment of rows, and marches down the segment in
// chunks of FR = 4 rows: one thread per site of the chunk.  Per chunk f
//   1. TMA (cp.async.bulk.tensor.3d, box {68, 4, C}, zero fill outside the lattice) has put the
//      raw inputs of chunk f (+2 halo columns each side) into a 2-stage smem buffer;
//   2. every thread turns its raw site into the two stage fields and writes them into two
//      16-row smem rings (the x-halo columns are done by 16 extra threads);
//   3. __syncthreads; thread 0 re-arms the stage with the TMA of chunk f+2;
//   4. every thread evaluates both radius-2 stencils of its site in chunk f-1 from the rings
//      (rows f-1 +- 2 are there), stores the results with coalesced 64-wide row stores and
//      contributes to the row-segment partial sums of the canonical tree.
// No y-halo is ever re-read from HBM except one warm-up chunk per segment end.
#pragma once
#include <cuda.h>

#include "ss_theory.cuh"

namespace ss {

constexpr int FW = SEG;             // strip width = row segment of the reduction tree
constexpr int FR = 4;               // rows per chunk
constexpr int FWP = FW + 2 * HALO;  // ring width
constexpr int RING = 16;            // ring rows (4 chunks: f-2, f-1, f and the one being filled)
constexpr int NST = 2;              // TMA stages
constexpr int FTHREADS = FW * FR;
constexpr int KX = 0, KY = 1;

template <typename real>
struct FlowArgs {
  alignas(64) CUtensorMap tm[4];  // phi, v, a1, a2 as (x, y, batch*C) tensors
  real* out0;                     // X: a1    Y: phi'
  real* out1;                     // X: a2    Y: v'
  double* part0;                  // X: e     Y: ke     [batch][Ny][nseg]
  double* part1;                  // X: q
  const LatticeState* state;
  const double* Bb;               // [batch] Zeeman field per lattice
  int Nx, Ny, nseg, cps;          // cps = chunks per segment
  long long plane;                // Nx*Ny
  real hdt, dt, qdt2, hdt2;       // dt/2, dt, dt^2/4, dt^2/2
  real sdt2, sdt;                 // dt^2/6, dt/6
  real i12h, i12h2;               // 1/(12h), 1/(12h^2)
  real kappa, K, lambda;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok = 0;
  while (!ok) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, int x, int y, int z,
                                            uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_u32(dst)),
      "l"(tm), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
      : "memory");
}

template <int THEORY, typename real, int KIND>
struct FlowCfg {
  static constexpr int C = TheoryOf<THEORY, real>::type::C;
  static constexpr int NARR = KIND == KX ? 2 : 4;
  static constexpr int XPAD = 16 / (int)sizeof(real);            // box starts 16-byte aligned
  static constexpr int RAWW = FW + 2 * XPAD;                     // staged width (>= FWP)
  static constexpr int BOXB = C * FR * RAWW * (int)sizeof(real); // bytes one TMA box delivers
  static constexpr int ARRB = (BOXB + 127) / 128 * 128;          // 128-byte aligned slot
  static constexpr int STAGEB = NARR * ARRB;
  static constexpr int RINGN = C * RING * FWP;                   // elements of one ring
  static constexpr int OFF_RING = NST * STAGEB;
  static constexpr int OFF_RED = OFF_RING + 2 * RINGN * (int)sizeof(real);
  static constexpr int OFF_BAR = OFF_RED + 2 * FR * (int)sizeof(double);
  static constexpr int SMEM = OFF_BAR + NST * 8;
  static constexpr int MINB = SMEM <= 110 * 1024 ? 2 : 1;        // CTAs per SM (227 KB)
};

template <int THEORY, typename real, int KIND>
__global__ void __launch_bounds__(FTHREADS, FlowCfg<THEORY, real, KIND>::MINB)
    flow_kernel(const __grid_constant__ FlowArgs<real> p) {
  using Th = typename TheoryOf<THEORY, real>::type;
  using Cfg = FlowCfg<THEORY, real, KIND>;
  constexpr int C = Cfg::C;
  extern __shared__ __align__(128) unsigned char smem[];
  real* ringA = reinterpret_cast<real*>(smem + Cfg::OFF_RING);  // X: phi    Y: phi3
  real* ringB = ringA + Cfg::RINGN;                             // X: phi2   Y: phi4
  double* red = reinterpret_cast<double*>(smem + Cfg::OFF_RED); // [2][FR]
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + Cfg::OFF_BAR);

  const int tid = threadIdx.x;
  const int tx = tid & (FW - 1), r = tid >> 6, lane = tid & 31;
  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z, x0 = blockIdx.x * FW;
  const int NC = (Ny + FR - 1) / FR;
  const int cs = blockIdx.y * p.cps, ce = min(cs + p.cps, NC);  // stencil chunks [cs, ce)
  const int f0 = max(cs - 1, 0), f1 = min(ce, NC - 1);          // fill chunks [f0, f1]
  const bool vz = KIND == KY ? (p.state[b].v_is_zero != 0) : false;
  const real Bz = real(p.Bb[b]);

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // an arrested step needs neither v (vh = 0) nor a2 (a2 := a1)
  auto issue = [&](int f) {
    unsigned char* st = smem + ((f - f0) % NST) * Cfg::STAGEB;
    uint64_t* bar = &full[(f - f0) % NST];
    const int narr = KIND == KX ? 2 : (vz ? 2 : 4);
    mbar_expect_tx(bar, (uint32_t)(narr * Cfg::BOXB));
#pragma unroll
    for (int a = 0; a < Cfg::NARR; ++a) {
      if (KIND == KY && vz && (a == 1 || a == 3)) continue;
      tma_load_3d(st + a * Cfg::ARRB, &p.tm[a], x0 - Cfg::XPAD, f * FR, b * C, bar);
    }
  };
  if (tid == 0)
    for (int f = f0; f < f0 + NST && f <= f1; ++f) issue(f);

  // raw site -> the two stage fields in the rings; returns the pointwise RK4 data of the site
  real keep_new[2 * C], keep_old[2 * C];
#pragma unroll
  for (int c = 0; c < 2 * C; ++c) keep_new[c] = keep_old[c] = real(0);

  auto fill_site = [&](const unsigned char* st, int f, int row, int lx, bool keep) {
    const int gx = x0 - HALO + lx, gy = f * FR + row;
    const bool inter = gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO;
    constexpr int RW = Cfg::RAWW;
    const int ro = row * RW + lx + (Cfg::XPAD - HALO);
    const real* rphi = reinterpret_cast<const real*>(st);
    const real* rvel = reinterpret_cast<const real*>(st + Cfg::ARRB);
    real ph[C], A[C], Bf[C];
#pragma unroll
    for (int c = 0; c < C; ++c) ph[c] = rphi[c * FR * RW + ro];
    if (KIND == KX) {
#pragma unroll
      for (int c = 0; c < C; ++c) {
        A[c] = ph[c];
        Bf[c] = ph[c] + p.hdt * rvel[c * FR * RW + ro];
      }
      Th::project_field(Bf);
    } else {
      const real* ra1 = reinterpret_cast<const real*>(st + 2 * Cfg::ARRB);
      const real* ra2 = reinterpret_cast<const real*>(st + 3 * Cfg::ARRB);
      real k0[C], k1[C];
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const real a1 = ra1[c * FR * RW + ro];
        const real vh = vz ? real(0) : rvel[c * FR * RW + ro];
        const real a2 = vz ? a1 : ra2[c * FR * RW + ro];
        A[c] = (ph[c] + p.hdt * vh) + p.qdt2 * a1;
        const real base = ph[c] + p.dt * vh;
        Bf[c] = base + p.hdt2 * a2;
        k0[c] = base + p.sdt2 * (a1 + a2);
        k1[c] = vh + p.sdt * (a1 + real(2) * a2);
      }
      Th::project_field(A);
      Th::project_field(Bf);
      if (keep) {
#pragma unroll
        for (int c = 0; c < C; ++c) { keep_new[c] = k0[c]; keep_new[C + c] = k1[c]; }
      }
    }
    const int wo = (gy & (RING - 1)) * FWP + lx;
#pragma unroll
    for (int c = 0; c < C; ++c) {
      ringA[c * RING * FWP + wo] = inter ? A[c] : ph[c];
      ringB[c * RING * FWP + wo] = inter ? Bf[c] : ph[c];
    }
  };

  for (int f = f0; f <= ce; ++f) {
    if (f <= f1) {
      const int k = f - f0;
      const unsigned char* st = smem + (k % NST) * Cfg::STAGEB;
      mbar_wait(&full[k % NST], (uint32_t)((k / NST) & 1));
      fill_site(st, f, r, tx + HALO, true);
      if (tid < 4 * FR) {
        const int q = tid & 3;
        fill_site(st, f, tid >> 2, q < 2 ? q : FW + q, false);
      }
    }
    __syncthreads();
    if (tid == 0 && f + NST <= f1) issue(f + NST);

    const int sc = f - 1;
    if (sc >= cs && sc < ce) {
      const int gx = x0 + tx, gy = sc * FR + r;
      const bool active = gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO;
      double s0 = 0.0, s1 = 0.0;
      if (active) {
        int ro[5];
#pragma unroll
        for (int d = 0; d < 5; ++d) ro[d] = ((gy + d - 2) & (RING - 1)) * FWP + tx + HALO;
        auto TA = [&](int c, int dy, int dx) -> real { return ringA[c * RING * FWP + ro[dy + 2] + dx]; };
        auto TB = [&](int c, int dy, int dx) -> real { return ringB[c * RING * FWP + ro[dy + 2] + dx]; };
        const long long o = (long long)b * C * p.plane + (long long)gy * Nx + gx;
        real aA[C], aB[C];
        Th::accel(TA, p, Bz, aA);
        if (KIND == KX) {
#pragma unroll
          for (int c = 0; c < C; ++c) p.out0[o + c * p.plane] = aA[c];
          real e, q;
          EdgeW w(gx, gy, Nx, Ny);
          Th::densities(TA, p, Bz, w, e, q);
          s0 = double(e);
          s1 = double(q);
          Th::accel(TB, p, Bz, aB);
#pragma unroll
          for (int c = 0; c < C; ++c) p.out1[o + c * p.plane] = aB[c];
        } else {
          Th::accel(TB, p, Bz, aB);
          real fn[C], u[C];
#pragma unroll
          for (int c = 0; c < C; ++c) {
            fn[c] = keep_old[c] + p.sdt2 * aA[c];
            u[c] = keep_old[C + c] + p.sdt * (real(2) * aA[c] + aB[c]);
          }
          Th::project_field(fn);
          Th::project_velocity(u, fn);
          real v2 = real(0);
#pragma unroll
          for (int c = 0; c < C; ++c) {
            p.out0[o + c * p.plane] = fn[c];
            p.out1[o + c * p.plane] = u[c];
            v2 += u[c] * u[c];
          }
          s0 = 0.5 * double(v2);
        }
      }
      // row-segment partial sums: aligned pairwise tree over the 64 sites of (row, strip)
      s0 = warp_tree(s0);
      if (KIND == KX) s1 = warp_tree(s1);
      if (lane == 0 && tx >= 32) {
        red[r] = s0;
        if (KIND == KX) red[FR + r] = s1;
      }
      asm volatile("bar.sync %0, 64;" ::"r"(1 + r) : "memory");
      if (tx == 0 && gy < Ny) {
        const long long po = ((long long)b * Ny + gy) * p.nseg + blockIdx.x;
        p.part0[po] = s0 + red[r];
        if (KIND == KX) p.part1[po] = s1 + red[FR + r];
      }
    }
#pragma unroll
    for (int c = 0; c < 2 * C; ++c) keep_old[c] = keep_new[c];
  }
}

}  // namespace ss
