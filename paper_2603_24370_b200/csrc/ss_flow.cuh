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
//   flow_kernel<THEORY, real, KV>  "V": the whole one-gradient-per-step (velocity Verlet, DESIGN
//       R15) step: reads phi, v, a -> writes phi', v', a', E/Q/KE partials
//       w = vh + dt/2 a, phi' = R(phi + dt w), a' = -Pi G(phi'), v' = Pi(w + dt/2 a')
//
// A CTA owns a strip of FW = 64 columns and a segment of rows, and marches down the segment in
// chunks of FR = 4 rows; a thread owns SPT vertically adjacent sites of the chunk (fp32 chiral
// magnet: VEC = 2 horizontally adjacent columns, computed with packed f2 arithmetic).  Per chunk f
//   1. TMA (cp.async.bulk.tensor.3d, box {64 + 2 XPAD, 4, C}, zero fill outside the lattice, box
//      start 16-byte aligned) has put the raw inputs of chunk f into an NST-stage smem buffer;
//   2. every thread turns its raw sites into the stage field(s) and writes them into smem rings
//      of RING rows x 68 columns (the 16 x-halo sites of the chunk are done by a few threads);
//   3. __syncthreads; thread 0 re-arms the freed stage with the TMA of chunk f + NST;
//   4. every thread evaluates the radius-2 stencil(s) of its sites in chunk f-1 from the rings
//      (rows f-1 +- 2 are there; the sites of a thread share their column through registers),
//      does the pointwise integrator algebra with data kept in registers since step 2, stores the
//      results with coalesced row stores and contributes to the row-segment partial sums of the
//      canonical tree (warp xor-shuffle tree, then low half + high half after the next barrier).
// No y-halo is ever re-read from HBM except one warm-up chunk per segment end.
// A launch covers the y-segments [seg0, seg0 + gridDim.y): all of them, or -- on large single
// lattices -- one row slab of the step's graph, in which X of a slab starts as soon as Y of the
// slab and of its two neighbours is done (ss_api.cu plan_slabs).
#pragma once
#include <cuda.h>

#include <type_traits>

#include "ss_theory.cuh"

namespace ss {

constexpr int FW = SEG;             // strip width = row segment of the reduction tree
constexpr int FR = 4;               // rows per chunk
constexpr int FWP = FW + 2 * HALO;  // ring width
constexpr int KX = 0, KY = 1, KV = 2, KXD = 3;  // KXD: kernel X with phi delivered into ring A (fp64)

template <typename real>
struct FlowArgs {
  alignas(64) CUtensorMap tm[4];  // phi, v, a1 (V: a), a2 as (x, y, batch*C) tensors
  real* out0;                     // X: a1    Y, V: phi'
  real* out1;                     // X: a2    Y, V: v'
  real* out2;                     //          V: a'
  double* part0;                  // X, V: e  Y: ke     [batch][Ny][nseg]
  double* part1;                  // X, V: q
  double* part2;                  // V: ke
  const LatticeState* state;
  const double* Bb;               // [batch] Zeeman field per lattice
  int Nx, Ny, nseg, cps;          // cps = chunks per segment
  int seg0;                       // first y-segment of this launch (row slabs, ss_api.cu)
  long long plane;                // Nx*Ny
  real hdt, dt, qdt2, hdt2;       // dt/2, dt, dt^2/4, dt^2/2
  real sdt2, sdt;                 // dt^2/6, dt/6
  real i12h, i12h2;               // 1/(12h), 1/(12h^2)
  real kappa, K, lambda;
  real lap0, lap1, lap2;          // 60, 16, 1 / (12 h^2)
  real dm1, dm2, K2;              // 2 kappa (8, 1) / (12 h); 2 K
  real jA, jB, hk, qs;            // J1/4h^2, J2/4h^2, kappa/(12h), 1/(4 pi (12h)^2)
  real dk[6];                     // kappa/(12h) * (d_x, d_y)   (general DMI table)
  real bs_k2, bs_mu2;             // baby Skyrme: kappa^2, mu^2
  int bs_pot, bs_potN;            //              potential, N of the Z_N one
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

__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap* tm, int x, int y, int z) {
  asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global [%0, {%1, %2, %3}];" ::"l"(tm), "r"(x),
               "r"(y), "r"(z)
               : "memory");
}

// Shape of the march, per kernel (measured on B200): 2 vertically adjacent
// sites per thread, 14-row rings (chunks f-1, f, f+1 and two rows of f-2 are live, one barrier
// per chunk), 3 CTAs per SM; two TMA stages in X and V, one in Y (so that the third CTA fits).
// fp32 chiral magnet: 2 horizontally adjacent columns per thread (packed f2), 1 row, 5 CTAs/SM.
constexpr int SPT_F64 = 2, SPT_F32V = 1;
constexpr int RING_ROWS = 14;
constexpr int MINB_F64 = 3, MINB_F32V = 5;

template <int THEORY, typename real, int KIND>
struct FlowCfg {
  static constexpr int C = TheoryOf<THEORY, real>::type::C;
  // columns per thread: 2 (packed f2 arithmetic) for the fp32 chiral magnet, else 1
  static constexpr int VEC = (sizeof(real) == 4 && THEORY != kAH) ? 2 : 1;
  static constexpr int SPT = VEC == 2 ? SPT_F32V : SPT_F64;
  static constexpr int ROWT = FR / SPT;                          // thread rows
  static constexpr int LX = FW / VEC;                            // threads per row
  static constexpr int THREADS = LX * ROWT;
  static constexpr int RING = RING_ROWS;
  // KXD (fp64 chiral magnet, schedules without row slabs): kernel X's ring A is phi itself, so TMA
  // delivers phi straight into a 16-row ring A (four chunk slots, one {68, 4, 1} box per
  // component) and only v passes through a single stage buffer; the CTA shrinks from 72 to 55 KB
  // and 116 registers: 4 CTAs per SM.  Same arithmetic, bitwise the same results as KX.
  static constexpr bool ISX = KIND == KX || KIND == KXD;
  static constexpr bool DIRECT = KIND == KXD;
  static constexpr int RINGA = DIRECT ? 16 : RING;               // rows of ring A
  static constexpr int NST = (KIND == KY || DIRECT) ? 1 : 2;     // TMA stages
  static constexpr int XPAD = 16 / (int)sizeof(real);            // box starts 16-byte aligned
  static constexpr int RAWW = FW + 2 * XPAD;                     // staged width (>= FWP)
  static constexpr int BOXB = C * FR * RAWW * (int)sizeof(real); // bytes one TMA box delivers
  static constexpr int ARRB = (BOXB + 127) / 128 * 128;          // 128-byte aligned slot
  static constexpr int NARR = ISX ? 2 : (KIND == KY ? 4 : 3);  // phi, v (, a1 (, a2))
  static constexpr int NRING = KIND == KV ? 1 : 2;
  static constexpr int STAGEB = (DIRECT ? 1 : NARR) * ARRB;      // DIRECT: v only
  static constexpr int OFF_RING = NST * STAGEB;
  static constexpr int RP = RING * FWP;                          // elements of one plane of ring B
  static constexpr int RPA = RINGA * FWP;                        // ... of ring A
  static constexpr int RINGN = C * RP;                           // elements of ring B
  static constexpr int OFF_RED = OFF_RING + (C * RPA + (NRING - 1) * RINGN) * (int)sizeof(real);
  static constexpr int OFF_BAR = OFF_RED + 2 * 3 * FR * 2 * (int)sizeof(double);
  static constexpr int SMEM = OFF_BAR + NST * 8;
  static constexpr int FITB = (227 * 1024) / (SMEM + 1024);      // CTAs per SM that fit
  static constexpr int WANTB = VEC == 2 ? MINB_F32V : (DIRECT ? MINB_F64 + 1 : MINB_F64);
  static_assert(!DIRECT || sizeof(real) == 8, "KXD is an fp64 kernel");
  static constexpr int MINB = FITB < 1 ? 1 : (FITB < WANTB ? FITB : WANTB);
  static_assert(FR % SPT == 0 && RING >= 3 * FR + 2, "ring too small");
  static_assert(!DIRECT || (RAWW == FWP && RINGA == 4 * FR && ARRB == BOXB), "DIRECT layout");
  __device__ __forceinline__ static int ring_row_a(int gy) {
    return DIRECT ? (gy & (RINGA - 1)) : ring_row(gy);
  }
  __device__ __forceinline__ static int ring_row(int gy) {       // gy >= -RING
    return (RING & (RING - 1)) == 0 ? (gy & (RING - 1)) : (int)((unsigned)(gy + RING) % RING);
  }
};

// combined aligned pairwise tree of two quantities over the 32 lanes: even lanes end with the
// sum of a, odd lanes with the sum of b (5 shuffles instead of 10; IEEE addition commutes)
__device__ __forceinline__ double warp_tree2(double a, double b, int lane) {
  const bool odd = lane & 1;
  const double give = odd ? a : b;
  double mine = (odd ? b : a) + __shfl_xor_sync(0xffffffffu, give, 1);
#pragma unroll
  for (int o = 2; o < 32; o <<= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
  return mine;
}

// the value a thread computes with: one site, or two side by side
template <typename real, int VEC> struct VecOf { using type = real; };
template <> struct VecOf<float, 2> { using type = f2; };
template <typename V, typename real> __device__ __forceinline__ V vload(const real* q) { return V(*q); }
template <> __device__ __forceinline__ f2 vload<f2, float>(const float* q) {
  return f2(*reinterpret_cast<const float2*>(q));
}
template <typename real> __device__ __forceinline__ void vstore(real* q, real v) { *q = v; }
__device__ __forceinline__ void vstore(float* q, f2 v) { *reinterpret_cast<float2*>(q) = v.v; }
__device__ __forceinline__ double vsum(double v) { return v; }
__device__ __forceinline__ double vsum(float v) { return double(v); }
__device__ __forceinline__ double vsum(f2 v) { return double(v.v.x) + double(v.v.y); }  // tree level 1
__device__ __forceinline__ float vlo(f2 v) { return v.v.x; }
__device__ __forceinline__ float vhi(f2 v) { return v.v.y; }
template <typename T> __device__ __forceinline__ T vlo(T v) { return v; }
template <typename T> __device__ __forceinline__ T vhi(T v) { return v; }

// halo weights of two side-by-side sites (DESIGN R3)
struct EdgeW2 {
  EdgeW a, b;
  __device__ __forceinline__ EdgeW2(int gx, int gy, int Nx, int Ny) : a(gx, gy, Nx, Ny), b(gx + 1, gy, Nx, Ny) {}
  __device__ __forceinline__ f2 wx(int s) const { return f2(float(a.x[s]), float(b.x[s])); }
  __device__ __forceinline__ f2 wy(int s) const { return f2(float(a.y[s]), float(b.y[s])); }
};

template <int THEORY, typename real, int KIND>
__global__ void __launch_bounds__(FlowCfg<THEORY, real, KIND>::THREADS,
                                  FlowCfg<THEORY, real, KIND>::MINB)
    flow_kernel(const __grid_constant__ FlowArgs<real> p) {
  using Cfg = FlowCfg<THEORY, real, KIND>;
  constexpr int C = Cfg::C, RP = Cfg::RP, RPA = Cfg::RPA, SPT = Cfg::SPT, NST = Cfg::NST, VEC = Cfg::VEC;
  using vreal = typename VecOf<real, VEC>::type;
  using Th = typename TheoryOf<THEORY, vreal>::type;
  constexpr int NQ = Cfg::ISX ? 2 : (KIND == KY ? 1 : 3);  // partial-sum quantities
  extern __shared__ __align__(128) unsigned char smem[];
  real* ringA = reinterpret_cast<real*>(smem + Cfg::OFF_RING);  // X: phi    Y: phi3   V: phi'
  real* ringB = ringA + (Cfg::NRING - 1) * C * RPA;             // X: phi2   Y: phi4
  double* red = reinterpret_cast<double*>(smem + Cfg::OFF_RED); // [2 parity][3 q][FR][2 halves]
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + Cfg::OFF_BAR);

  const int tid = threadIdx.x;
  const int tx = (tid % Cfg::LX) * VEC, r0 = (tid / Cfg::LX) * SPT, lane = tid & 31;  // columns tx..tx+VEC-1, rows r0..r0+SPT-1
  const int Nx = p.Nx, Ny = p.Ny;
  const int b = blockIdx.z, x0 = blockIdx.x * FW;
  const int NC = (Ny + FR - 1) / FR;
  const int cs = (blockIdx.y + p.seg0) * p.cps, ce = min(cs + p.cps, NC);  // stencil chunks [cs, ce)
  const int f0 = max(cs - 1, 0), f1 = min(ce, NC - 1);          // fill chunks [f0, f1]
  const bool vz = !Cfg::ISX ? (p.state[b].v_is_zero != 0) : false;
  const vreal Bz = vreal(real(p.Bb[b]));

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
    const int narr = Cfg::ISX ? 2 : (KIND == KY ? (vz ? 2 : 4) : (vz ? 2 : 3));
    mbar_expect_tx(bar, (uint32_t)(narr * Cfg::BOXB));
    if constexpr (Cfg::DIRECT) {  // phi: one {68, 4, 1} box per component into the chunk's ring slot
#pragma unroll
      for (int c = 0; c < C; ++c)
        tma_load_3d(ringA + c * RPA + Cfg::ring_row_a(f * FR) * FWP, &p.tm[2], x0 - Cfg::XPAD, f * FR,
                    b * C + c, bar);
      tma_load_3d(st, &p.tm[1], x0 - Cfg::XPAD, f * FR, b * C, bar);
      return;
    }
#pragma unroll
    for (int a = 0; a < Cfg::NARR; ++a) {
      if (!Cfg::ISX && vz && (a == 1 || a == 3)) continue;
      tma_load_3d(st + a * Cfg::ARRB, &p.tm[a], x0 - Cfg::XPAD, f * FR, b * C, bar);
    }
    // Kernel Y has a single stage (17 % of its stall samples wait for it): the boxes of the chunk
    // after this one are pulled into the L2 now, so that their TMA load, issued one chunk later,
    // has the short latency.  Y alone 0.458 -> 0.444 ms, fp32 0.243 -> 0.230; no gain for X and V
    // (two stages), and nothing at two chunks ahead.
    if (KIND == KY && f + 1 <= f1) {
#pragma unroll
      for (int a = 0; a < Cfg::NARR; ++a) {
        if (vz && (a == 1 || a == 3)) continue;
        tma_prefetch_3d(&p.tm[a], x0 - Cfg::XPAD, (f + 1) * FR, b * C);
      }
    }
  };
  if (tid == 0)
    for (int f = f0; f < f0 + NST && f <= f1; ++f) issue(f);

  // pointwise RK4 data of the thread's sites, carried from their fill to their stencil (Y):
  // [0,C) = (phi + dt vh) + dt^2/6 (a1 + a2),  [C,2C) = vh + dt/6 (a1 + 2 a2)
  vreal keep_new[SPT][2 * C], keep_old[SPT][2 * C];
#pragma unroll
  for (int k = 0; k < SPT; ++k)
#pragma unroll
    for (int c = 0; c < 2 * C; ++c) keep_new[k][c] = keep_old[k][c] = vreal(real(0));

  // raw site (row, lx) of chunk f -> the two stage fields in the rings
  // (edge_tag = false_type: the caller knows the site is interior, no test is compiled)
  auto fill_site = [&](const unsigned char* st, int f, int row, int lx, vreal* keep, auto edge_tag) {
    constexpr int RW = Cfg::RAWW;
    const int gx = x0 - HALO + lx, gy = f * FR + row;
    const bool inter = !decltype(edge_tag)::value ||
                       (gx >= HALO && gx < Nx - HALO && gy >= HALO && gy < Ny - HALO);
    const int ro = row * RW + lx + (Cfg::XPAD - HALO);
    const real* rphi = reinterpret_cast<const real*>(st);
    const real* rvel = reinterpret_cast<const real*>(st + Cfg::ARRB);
    vreal A[C], Bf[C];
    if constexpr (Cfg::DIRECT) {  // phi is in ring A already (TMA); the stage holds v only
      const int ao = Cfg::ring_row_a(gy) * FWP + lx;
#pragma unroll
      for (int c = 0; c < C; ++c) A[c] = Bf[c] = vload<vreal>(ringA + c * RPA + ao);
      if (inter) {
#pragma unroll
        for (int c = 0; c < C; ++c) Bf[c] = A[c] + p.hdt * vload<vreal>(rphi + c * FR * RW + ro);
        Th::project_field(Bf);
      }
      const int wb = Cfg::ring_row(gy) * FWP + lx;
#pragma unroll
      for (int c = 0; c < C; ++c) vstore(ringB + c * RP + wb, Bf[c]);
      return;
    }
#pragma unroll
    for (int c = 0; c < C; ++c) A[c] = Bf[c] = vload<vreal>(rphi + c * FR * RW + ro);
    if (inter) {  // halo sites of every stage field are the frozen halo
      if (Cfg::ISX) {
#pragma unroll
        for (int c = 0; c < C; ++c) Bf[c] = A[c] + p.hdt * vload<vreal>(rvel + c * FR * RW + ro);
        Th::project_field(Bf);
      } else if (KIND == KV) {
        const real* ra = reinterpret_cast<const real*>(st + 2 * Cfg::ARRB);
#pragma unroll
        for (int c = 0; c < C; ++c) {
          const vreal vh = vz ? vreal(real(0)) : vload<vreal>(rvel + c * FR * RW + ro);
          const vreal w = vh + p.hdt * vload<vreal>(ra + c * FR * RW + ro);
          A[c] = A[c] + p.dt * w;
          if (keep) keep[c] = w;
        }
        Th::project_field(A);
      } else {
        const real* ra1 = reinterpret_cast<const real*>(st + 2 * Cfg::ARRB);
        const real* ra2 = reinterpret_cast<const real*>(st + 3 * Cfg::ARRB);
#pragma unroll
        for (int c = 0; c < C; ++c) {
          const vreal ph = A[c];
          const vreal a1 = vload<vreal>(ra1 + c * FR * RW + ro);
          const vreal vh = vz ? vreal(real(0)) : vload<vreal>(rvel + c * FR * RW + ro);
          const vreal a2 = vz ? a1 : vload<vreal>(ra2 + c * FR * RW + ro);
          A[c] = (ph + p.hdt * vh) + p.qdt2 * a1;
          const vreal base = ph + p.dt * vh;
          Bf[c] = base + p.hdt2 * a2;
          if (keep) {
            keep[c] = base + p.sdt2 * (a1 + a2);
            keep[C + c] = vh + p.sdt * (a1 + vreal(real(2)) * a2);
          }
        }
        Th::project_field(A);
        Th::project_field(Bf);
      }
    }
    const int wo = Cfg::ring_row(gy) * FWP + lx;  // not DIRECT: both rings have RING rows
#pragma unroll
    for (int c = 0; c < C; ++c) {
      vstore(ringA + c * RPA + wo, A[c]);
      if (KIND != KV) vstore(ringB + c * RP + wo, Bf[c]);
    }
  };

  // row-segment partial sums of chunk sc (written by the two warps of each row into `red`)
  auto flush_partials = [&](int sc, int par) {
    if (tid < NQ * FR) {
      const int q = tid / FR, row = tid % FR, gy = sc * FR + row;
      if (gy < Ny) {
        const double* rr = red + ((par * 3 + q) * FR + row) * 2;
        double* dst = q == 0 ? p.part0 : (q == 1 ? p.part1 : p.part2);
        dst[((long long)b * Ny + gy) * p.nseg + blockIdx.x] = rr[0] + rr[1];
      }
    }
  };

  const int gx = x0 + tx;  // first column of the thread (pairs never straddle the halo: Nx % 4 == 0)
  const bool xin = gx >= HALO && gx < Nx - HALO;
  const bool xedge = gx < 2 * HALO || gx >= Nx - 2 * HALO;

  // One iteration of the march: fill chunk f, barrier, stencils of chunk f - 1.  EDGE = false is
  // the steady state of a strip away from the lattice edge: chunk f is filled and chunk f - 1
  // evaluated, every site involved is interior and at least 4 sites from the halo, so no
  // per-site test exists and the sites of a thread are straight-line code that the compiler
  // interleaves.  EDGE = true keeps every test (edge strips, first / last chunks of a segment).
  auto iteration = [&](const int f, auto edge_tag) {
    constexpr bool EDGE = decltype(edge_tag)::value;
    if (!EDGE || f <= f1) {
      const int k = f - f0;
      const unsigned char* st = smem + (k % NST) * Cfg::STAGEB;
      mbar_wait(&full[k % NST], (uint32_t)((k / NST) & 1));
#pragma unroll
      for (int k2 = 0; k2 < SPT; ++k2) fill_site(st, f, r0 + k2, tx + HALO, keep_new[k2], edge_tag);
      if (tid < 4 * FR / VEC) {  // the x-halo columns 0, 1, FW+2, FW+3 of the chunk's rows
        const int q = tid % (4 / VEC) * VEC;
        fill_site(st, f, tid / (4 / VEC), q < 2 ? q : FW + q, nullptr, edge_tag);
      }
    }
    __syncthreads();
    if (tid == 0 && f + NST <= f1) issue(f + NST);

    const int sc = f - 1;
    if (sc - 1 >= cs && sc - 1 < ce) flush_partials(sc - 1, (f - 1) & 1);
    if (!EDGE || (sc >= cs && sc < ce)) {
      const int gy0 = sc * FR + r0;
      // ring offsets of rows gy0-2 .. gy0+SPT+1 at the thread's column
      int rw[SPT + 4], rwa[SPT + 4];  // ring B / ring A (the same unless DIRECT)
#pragma unroll
      for (int j = 0; j < SPT + 4; ++j) {
        rw[j] = Cfg::ring_row(gy0 - HALO + j) * FWP + tx + HALO;
        rwa[j] = Cfg::ring_row_a(gy0 - HALO + j) * FWP + tx + HALO;
      }
      // tile accessor: component c, ring row slot j, x offset dx of the thread's first column;
      // with two columns per thread the odd offsets are recombined from the aligned pairs
      auto tile = [&](const real* ring, const int rp, const vreal (&colr)[C][SPT + 4],
                      const int (&rwr)[SPT + 4], int c, int j, int dx) -> vreal {
        if constexpr (VEC == 1) {
          return dx == 0 ? colr[c][j] : vreal(ring[c * rp + rwr[j] + dx]);
        } else {
          auto pr = [&](int dxe) -> vreal {
            return dxe == 0 ? colr[c][j] : vload<vreal>(ring + c * rp + rwr[j] + dxe);
          };
          if (dx == 0 || dx == 2 || dx == -2) return pr(dx);
          if (dx == 1) return vreal(vhi(pr(0)), vlo(pr(2)));
          return vreal(vhi(pr(-2)), vlo(pr(0)));
        }
      };
      double s0[SPT], s1[SPT], s2[SPT];
      bool act[SPT];
      vreal aA[SPT][C];
#pragma unroll
      for (int k = 0; k < SPT; ++k) {
        s0[k] = s1[k] = s2[k] = 0.0;
        act[k] = !EDGE || (xin && gy0 + k >= HALO && gy0 + k < Ny - HALO);
      }
      const long long o = (long long)b * C * p.plane + (long long)gy0 * Nx + gx;
      real* o0 = p.out0 + o;
      real* o1 = p.out1 + o;
      // The SPT sites of a thread share their column: its SPT+4 ring values per component are
      // loaded once into registers; only the x-neighbours are read per site.
      vreal col[C][SPT + 4];
      // Abelian Higgs: (12h)^2 DxDy A_c = D_y (D_x A_c) down the thread's column: one eq. (1)
      // numerator per ring row (4 loads) shared by the SPT sites, instead of 16 loads per site
      [[maybe_unused]] vreal xy[SPT][2];
      [[maybe_unused]] auto mixed = [&](const real* ring, const int rp, const int (&rwr)[SPT + 4]) {
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          vreal dxr[SPT + 4];
#pragma unroll
          for (int j = 0; j < SPT + 4; ++j) {
            const real* q = ring + (2 + cc) * rp + rwr[j];
            dxr[j] = d1n<vreal>(vreal(q[-2]), vreal(q[-1]), vreal(q[1]), vreal(q[2]));
          }
#pragma unroll
          for (int k = 0; k < SPT; ++k)
            xy[k][cc] = d1n<vreal>(dxr[k], dxr[k + 1], dxr[k + 3], dxr[k + 4]);
        }
      };
      constexpr bool AHXY = THEORY == kAH && VEC == 1;
      // ---- ring A (X: phi -> a1, e, q    Y: phi3 -> a3)
      if constexpr (AHXY) mixed(ringA, RPA, rwa);
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int j = 0; j < SPT + 4; ++j) col[c][j] = vload<vreal>(ringA + c * RPA + rwa[j]);
#pragma unroll
      for (int k = 0; k < SPT; ++k) {
        if (act[k]) {
          const int gy = gy0 + k;
          auto TA = [&](int c, int dy, int dx) -> vreal { return tile(ringA, RPA, col, rwa, c, k + dy + 2, dx); };
          if (Cfg::ISX || KIND == KV) {
            vreal e, q;
            if (EDGE && (xedge || gy < 2 * HALO || gy >= Ny - 2 * HALO)) {
              if constexpr (AHXY) Th::accel_xy(TA, p, Bz, xy[k][0], xy[k][1], aA[k]);
              else Th::accel(TA, p, Bz, aA[k]);
              if constexpr (VEC == 2) Th::densities(TA, p, Bz, EdgeW2(gx, gy, Nx, Ny), e, q);
              else Th::densities(TA, p, Bz, EdgeW(gx, gy, Nx, Ny), e, q);
            } else {
              if constexpr (AHXY) Th::accel_densities_bulk_xy(TA, p, Bz, xy[k][0], xy[k][1], aA[k], e, q);
              else Th::accel_densities_bulk(TA, p, Bz, aA[k], e, q);
            }
            s0[k] = vsum(e);
            s1[k] = vsum(q);
            if (Cfg::ISX) {
#pragma unroll
              for (int c = 0; c < C; ++c) vstore(o0 + c * p.plane + k * Nx, aA[k][c]);
            } else {  // second half kick, tangent projection, KE
              vreal fn[C], u[C];
#pragma unroll
              for (int c = 0; c < C; ++c) {
                fn[c] = col[c][k + 2];
                u[c] = keep_old[k][c] + p.hdt * aA[k][c];
              }
              Th::project_velocity(u, fn);
              vreal v2 = vreal(real(0));
#pragma unroll
              for (int c = 0; c < C; ++c) {
                vstore(o0 + c * p.plane + k * Nx, fn[c]);
                vstore(o1 + c * p.plane + k * Nx, u[c]);
                vstore(p.out2 + o + c * p.plane + k * Nx, aA[k][c]);
                v2 += u[c] * u[c];
              }
              s2[k] = 0.5 * vsum(v2);
            }
          } else {
            if constexpr (AHXY) Th::accel_xy(TA, p, Bz, xy[k][0], xy[k][1], aA[k]);
            else Th::accel(TA, p, Bz, aA[k]);
          }
        }
      }
      // ---- ring B (X: phi2 -> a2    Y: phi4 -> a4, RK4 combine, projections, KE)
      if (KIND != KV) {
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int j = 0; j < SPT + 4; ++j) col[c][j] = vload<vreal>(ringB + c * RP + rw[j]);
        if constexpr (AHXY) mixed(ringB, RP, rw);
      }
#pragma unroll
      for (int k = 0; k < SPT; ++k) {
        if (KIND != KV && act[k]) {
          auto TB = [&](int c, int dy, int dx) -> vreal { return tile(ringB, RP, col, rw, c, k + dy + 2, dx); };
          vreal aB[C];
          if constexpr (AHXY) Th::accel_xy(TB, p, Bz, xy[k][0], xy[k][1], aB);
          else Th::accel(TB, p, Bz, aB);
          if (Cfg::ISX) {
#pragma unroll
            for (int c = 0; c < C; ++c) vstore(o1 + c * p.plane + k * Nx, aB[c]);
          } else {
            vreal fn[C], u[C];
#pragma unroll
            for (int c = 0; c < C; ++c) {
              fn[c] = keep_old[k][c] + p.sdt2 * aA[k][c];
              u[c] = keep_old[k][C + c] + p.sdt * (vreal(real(2)) * aA[k][c] + aB[c]);
            }
            Th::project_field(fn);
            Th::project_velocity(u, fn);
            vreal v2 = vreal(real(0));
#pragma unroll
            for (int c = 0; c < C; ++c) {
              vstore(o0 + c * p.plane + k * Nx, fn[c]);
              vstore(o1 + c * p.plane + k * Nx, u[c]);
              v2 += u[c] * u[c];
            }
            s0[k] = 0.5 * vsum(v2);
          }
        }
      }
      // aligned pairwise tree over the 32 sites of the warp; the two halves of the 64-site row
      // segment are added (low + high) by flush_partials after the next barrier
#pragma unroll
      for (int k = 0; k < SPT; ++k) {
        // VEC == 2: one warp holds the whole 64-site row segment (pair sums = tree level 1)
        double* rr = red + (((f & 1) * 3) * FR + r0 + k) * 2 + (VEC == 2 ? 0 : (tx >> 5));
        if (VEC == 2 && lane < NQ) rr[lane * FR * 2 + 1] = 0.0;
        if (Cfg::ISX || KIND == KV) {
          const double t = warp_tree2(s0[k], s1[k], lane);
          if (lane < 2) rr[lane * FR * 2] = t;
          if (KIND == KV) {
            const double t2 = warp_tree(s2[k]);
            if (lane == 0) rr[2 * FR * 2] = t2;
          }
        } else {
          const double t = warp_tree(s0[k]);
          if (lane == 0) rr[0] = t;
        }
      }
    }
#pragma unroll
    for (int k = 0; k < SPT; ++k)
#pragma unroll
      for (int c = 0; c < 2 * C; ++c) keep_old[k][c] = keep_new[k][c];
  };

  // strips whose columns (x-halo included) are all >= 4 sites from the lattice edge.  Abelian
  // Higgs keeps the one-site-at-a-time instance everywhere: its kernels sit at the 255-register
  // limit and interleaving two sites costs more than it hides (0.404 vs 0.392 ms at 2048^2).
  const bool inner_strip = THEORY != kAH && x0 >= 2 * HALO + HALO && x0 + FW + HALO <= Nx - 2 * HALO;
  for (int f = f0; f <= ce; ++f) {
    const bool steady = inner_strip && f <= f1 && f - 1 >= cs && f - 1 < ce &&
                        (f - 1) * FR >= 2 * HALO && f * FR + FR <= Ny - 2 * HALO;
    if (steady) iteration(f, std::false_type{});
    else iteration(f, std::true_type{});
  }
  __syncthreads();
  if (ce - 1 >= cs) flush_partials(ce - 1, ce & 1);
}

}  // namespace ss
