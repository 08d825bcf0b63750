// Resident flow kernel for lattices whose whole state fits in the shared memory of one
// thread-block cluster (BASELINE config 1, 64 x 64: the general path is launch-latency bound at
// 4 dependent kernels per step; the paper's own usage steps a small lattice a few steps at a
// time).  One cluster per lattice runs ALL k steps of ss_step(k) in one
// launch: the CTAs own contiguous row slabs, phi, v, a1, a2 and the stage fields live in shared
// memory, the two halo rows of a stage field are pushed into the neighbour CTAs through
// distributed shared memory, cluster.sync() replaces the kernel boundaries, and every CTA
// finishes the canonical reduction tree (DESIGN R10) and takes the arrest decision (PAPER.md:125
// eq. 4) redundantly, so nothing is broadcast.
//
// Per-site arithmetic is the flow kernels' own (the same CM<double> routines and the same
// expressions as fill_site / the RK4 combine in ss_flow.cuh, the same edge / bulk choice per
// site), and the reduction order is that of the flow kernels + row_reduce_kernel +
// finalize_kernel: fields, E, Q, KE and the arrest log are bitwise identical to the general
// path (tests/test_gpu_resident.py).  Chiral magnet (default DMI), fp64, Nx a multiple of 32.
#pragma once
#include <cooperative_groups.h>

#include "ss_flow.cuh"

namespace ss {

namespace cg = cooperative_groups;

constexpr int RES_THREADS = 512;
constexpr int RES_MAX_NY = 1024;

struct ResidentArgs {
  FlowArgs<double> k;  // per-site constants (tensor maps unused)
  double* phi;         // [batch][3][Ny][Nx] state in HBM: loaded once, stored once
  double* vel;
  double* a1;
  double* a2;
  LatticeState* state;
  long long* log;
  long long log_cap;
  const double* Bb;
  int rows;            // rows of the lattice per CTA (Ny = rows * cluster size)
  long long steps;
  double h2;
};

// doubles of dynamic shared memory per CTA
inline size_t resident_smem_doubles(int Nx, int Ny, int rows) {
  const size_t W = Nx, PS = (size_t)(rows + 4) * W, PO = (size_t)rows * W;
  return 4 * 3 * PS       // phi, S2, S3, S4 with two halo rows above and below
         + (2 * PO <= (size_t)RES_THREADS ? 4 : 3) * 3 * PO  // v, a1, a2 (+ a4 exchange, split mode)
         + 3 * (size_t)rows * (W / 32)  // per-warp partial sums of e, q, ke
         + 3 * (size_t)Ny               // all row sums of the lattice
         + 3 * 32 + 8;                  // y-tree scratch, totals
}

__global__ void __launch_bounds__(RES_THREADS, 1)
    resident_kernel(const __grid_constant__ ResidentArgs a) {
  using Th = CM<double>;
  const FlowArgs<double>& p = a.k;
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank(), CL = (int)cluster.num_blocks();
  const int Nx = p.Nx, Ny = p.Ny, W = Nx, RR = a.rows;
  const int b = blockIdx.y;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int PS = (RR + 4) * W, PO = RR * W, NW = W / 32;
  const int nsite = RR * W;
  const int gy0 = rank * RR;

  extern __shared__ __align__(16) double sm[];
  double* phi = sm;               // [3][RR+4][W], own rows at row offset 2
  double* S2 = phi + 3 * PS;
  double* S3 = S2 + 3 * PS;
  double* S4 = S3 + 3 * PS;
  double* vel = S4 + 3 * PS;      // [3][RR][W]
  double* A1 = vel + 3 * PO;
  double* A2 = A1 + 3 * PO;
  double* XB = A2 + 3 * PO;       // a4 handed from role 1 to role 0 (split mode only)
  double* wsum = XB + (2 * nsite <= RES_THREADS ? 3 * PO : 0);  // [3][RR][NW]
  double* rows_all = wsum + 3 * RR * NW;  // [3][Ny]
  double* ysh = rows_all + 3 * Ny;        // [3][32]
  double* tot = ysh + 3 * 32;     // [3] + flags

  const long long lat = (long long)b * 3 * p.plane;
  const double Bz = a.Bb[b];

  // ---- load the state (phi with its two halo rows on each side: halo SITES of the lattice
  // never change, so the pushes of the steps only ever refresh interior sites of those rows)
  for (int s = tid; s < (RR + 4) * W; s += RES_THREADS) {
    const int r = s / W - 2, x = s % W, gy = gy0 + r;
    if (gy < 0 || gy >= Ny) continue;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double v = a.phi[lat + c * p.plane + (long long)gy * Nx + x];
      phi[c * PS + (r + 2) * W + x] = v;
      S2[c * PS + (r + 2) * W + x] = v;
      S3[c * PS + (r + 2) * W + x] = v;
      S4[c * PS + (r + 2) * W + x] = v;
    }
  }
  for (int s = tid; s < nsite; s += RES_THREADS) {
    const int r = s / W, x = s - r * W;
    const long long o = (long long)(gy0 + r) * Nx + x;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      vel[c * PO + s] = a.vel[lat + c * p.plane + o];
      A1[c * PO + s] = a.a1[lat + c * p.plane + o];
      A2[c * PO + s] = a.a2[lat + c * p.plane + o];
    }
  }
  LatticeState st = a.state[b];
  bool vz = st.v_is_zero != 0;
  cluster.sync();  // every CTA's buffers exist before the first push

  // The two outermost own rows on each side of the slab are also the neighbour CTA's halo rows:
  // every value of a stage field is stored locally and, for those rows, pushed into the
  // neighbour's copy through distributed shared memory (made visible by the next cluster.sync()).
  double* up_base = rank > 0 ? cluster.map_shared_rank(sm, rank - 1) : nullptr;
  double* dn_base = rank + 1 < CL ? cluster.map_shared_rank(sm, rank + 1) : nullptr;
  auto put = [&](double* buf, int c, int r, int x, double v) {
    const int off = (int)(buf - sm) + c * PS + x;
    buf[c * PS + (r + 2) * W + x] = v;
    if (r < HALO && up_base) up_base[off + (RR + 2 + r) * W] = v;
    if (r >= RR - HALO && dn_base) dn_base[off + (r - (RR - HALO)) * W] = v;
  };
  auto active_site = [&](int x, int gy) {
    return x >= HALO && x < Nx - HALO && gy >= HALO && gy < Ny - HALO;
  };
  // per-warp sums (first five tree levels) of up to three quantities of the warp's 32 sites
  auto warp_sums = [&](int s, double v0, double v1, int nq, int q0) {
    const int r = s / W, x = s - r * W;
    v0 = warp_tree(v0);
    if (nq > 1) v1 = warp_tree(v1);
    if (lane == 0) {
      wsum[(q0 * RR + r) * NW + (x >> 5)] = v0;
      if (nq > 1) wsum[((q0 + 1) * RR + r) * NW + (x >> 5)] = v1;
    }
  };
  // row sums of e, q, ke of the CTA's rows -> every CTA's rows_all (x-tree: the flow kernels' low
  // + high halves, then row_reduce_kernel's aligned tree over the 64-site segments; Nx <= 1024:
  // at most 16 segments, one per lane, m = 1)
  auto row_sums = [&]() {
    const int nseg = (W + SEG - 1) / SEG;
    for (int r = wid; r < RR; r += RES_THREADS / 32) {
      double v[3];
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        const double lo = 2 * lane < NW ? wsum[(q * RR + r) * NW + 2 * lane] : 0.0;
        const double hi = 2 * lane + 1 < NW ? wsum[(q * RR + r) * NW + 2 * lane + 1] : 0.0;
        v[q] = lane < nseg ? lo + hi : 0.0;
      }
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
        for (int q = 0; q < 3; ++q) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
      }
      if (lane < CL) {
        double* dst = cluster.map_shared_rank(rows_all, lane);
#pragma unroll
        for (int q = 0; q < 3; ++q) dst[q * Ny + gy0 + r] = v[q];
      }
    }
  };
  // y-tree of finalize_kernel (1024 leaves = 32 groups of 32 rows; groups beyond Ny sum zeros)
  auto y_tree = [&]() {
    for (int g = wid; g < 32; g += RES_THREADS / 32) {
      double v[3] = {0.0, 0.0, 0.0};
      if (g * 32 < Ny) {
        const int row = g * 32 + lane;
#pragma unroll
        for (int q = 0; q < 3; ++q) v[q] = row < Ny ? rows_all[q * Ny + row] : 0.0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
          for (int q = 0; q < 3; ++q) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
        }
      }
      if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 3; ++q) ysh[q * 32 + g] = v[q];
      }
    }
  };

  // Work split.  With at most half as many sites as threads (64 x 64 on 16 CTAs: 256 sites, 512
  // threads) every site gets TWO threads: role 0 evaluates the first stage field of a phase
  // (phi3, then phi'), role 1 the second (phi4, then phi2'), each routine still run whole by one
  // thread on the same inputs, so nothing changes numerically.  Otherwise one thread does both.
  const bool split = 2 * nsite <= RES_THREADS;
  const int mask = split ? (tid < nsite ? 1 : (tid < 2 * nsite ? 2 : 0)) : 3;
  const int s0 = split ? (tid < nsite ? tid : tid - nsite) : tid;
  const int sstep = split ? 2 * nsite : RES_THREADS;  // split: exactly one site per thread
  const int send = mask ? nsite : 0;

  // ---- P1: stage fields phi3 (role 0), phi4 (role 1) of the own rows (fill_site of kernel Y)
  auto P1 = [&](bool vzz) {
    for (int s = s0; s < send; s += sstep) {
      const int r = s / W, x = s - r * W, gy = gy0 + r;
      double A[3], Bf[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) A[c] = Bf[c] = phi[c * PS + (r + 2) * W + x];
      if (active_site(x, gy)) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const double ph = A[c];
          const double a1 = A1[c * PO + s];
          const double vh = vzz ? 0.0 : vel[c * PO + s];
          const double a2 = vzz ? a1 : A2[c * PO + s];
          A[c] = (ph + p.hdt * vh) + p.qdt2 * a1;
          const double base = ph + p.dt * vh;
          Bf[c] = base + p.hdt2 * a2;
        }
        if (mask & 1) Th::project_field(A);
        if (mask & 2) Th::project_field(Bf);
      }
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        if (mask & 1) put(S3, c, r, x, A[c]);
        if (mask & 2) put(S4, c, r, x, Bf[c]);
      }
    }
  };
  // RK4 combine, projections, KE, phi2' of one site from a3 = aA, a4 = aB (kernel Y, X's fill)
  auto combine = [&](int s, int r, int x, const double (&aA)[3], const double (&aB)[3]) -> double {
    const int o = (r + 2) * W + x;
    double fn[3], u[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double ph = phi[c * PS + o];
      const double a1 = A1[c * PO + s];
      const double vh = vz ? 0.0 : vel[c * PO + s];
      const double a2 = vz ? a1 : A2[c * PO + s];
      const double base = ph + p.dt * vh;
      const double k0 = base + p.sdt2 * (a1 + a2);
      const double k1 = vh + p.sdt * (a1 + 2.0 * a2);
      fn[c] = k0 + p.sdt2 * aA[c];
      u[c] = k1 + p.sdt * (2.0 * aA[c] + aB[c]);
    }
    Th::project_field(fn);
    Th::project_velocity(u, fn);
    double v2 = 0.0, B2[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      put(phi, c, r, x, fn[c]);
      vel[c * PO + s] = u[c];
      v2 += u[c] * u[c];
      B2[c] = fn[c] + p.hdt * u[c];
    }
    Th::project_field(B2);
#pragma unroll
    for (int c = 0; c < 3; ++c) put(S2, c, r, x, B2[c]);
    return 0.5 * v2;
  };

  P1(vz);
  cluster.sync();
  for (long long it = 0; it < a.steps; ++it) {
    // ---- P2: a3 (role 0), a4 (role 1), then the combine
    if (split) {
      const int s = s0, r = s / W, x = s - r * W, gy = gy0 + r;
      const bool act = mask && active_site(x, gy);
      const int o = (r + 2) * W + x;
      double aA[3] = {0.0, 0.0, 0.0}, aB[3];
      if (act && mask == 1) {
        auto TA = [&](int c, int dy, int dx) -> double { return S3[c * PS + o + dy * W + dx]; };
        Th::accel(TA, p, Bz, aA);
      }
      if (act && mask == 2) {
        auto TB = [&](int c, int dy, int dx) -> double { return S4[c * PS + o + dy * W + dx]; };
        Th::accel(TB, p, Bz, aB);
#pragma unroll
        for (int c = 0; c < 3; ++c) XB[c * PO + s] = aB[c];
      }
      __syncthreads();
      if (mask == 1) {
        double ke = 0.0;
        if (act) {
#pragma unroll
          for (int c = 0; c < 3; ++c) aB[c] = XB[c * PO + s];
          ke = combine(s, r, x, aA, aB);
        } else {  // frozen halo: phi2' = phi there (the neighbours' copies of phi never change)
#pragma unroll
          for (int c = 0; c < 3; ++c) put(S2, c, r, x, phi[c * PS + o]);
        }
        warp_sums(s, ke, 0.0, 1, 2);
      }
    } else {
      for (int s = s0; s < send; s += sstep) {
        const int r = s / W, x = s - r * W, gy = gy0 + r;
        double ke = 0.0;
        if (active_site(x, gy)) {
          const int o = (r + 2) * W + x;
          auto TA = [&](int c, int dy, int dx) -> double { return S3[c * PS + o + dy * W + dx]; };
          auto TB = [&](int c, int dy, int dx) -> double { return S4[c * PS + o + dy * W + dx]; };
          double aA[3], aB[3];
          Th::accel(TA, p, Bz, aA);
          Th::accel(TB, p, Bz, aB);
          ke = combine(s, r, x, aA, aB);
        } else {
#pragma unroll
          for (int c = 0; c < 3; ++c) put(S2, c, r, x, phi[c * PS + (r + 2) * W + x]);
        }
        warp_sums(s, ke, 0.0, 1, 2);
      }
    }
    cluster.sync();

    // ---- P3: a1, e, q on phi' (role 0); a2 on phi2' (role 1)  (kernel X)
    for (int s = s0; s < send; s += sstep) {
      const int r = s / W, x = s - r * W, gy = gy0 + r;
      const bool act = active_site(x, gy);
      const int o = (r + 2) * W + x;
      if (mask & 1) {
        double e = 0.0, q = 0.0;
        if (act) {
          auto TA = [&](int c, int dy, int dx) -> double { return phi[c * PS + o + dy * W + dx]; };
          double aA[3];
          if (x < 2 * HALO || x >= Nx - 2 * HALO || gy < 2 * HALO || gy >= Ny - 2 * HALO) {
            Th::accel(TA, p, Bz, aA);
            Th::densities(TA, p, Bz, EdgeW(x, gy, Nx, Ny), e, q);
          } else {
            Th::accel_densities_bulk(TA, p, Bz, aA, e, q);
          }
#pragma unroll
          for (int c = 0; c < 3; ++c) A1[c * PO + s] = aA[c];
        }
        warp_sums(s, e, q, 2, 0);
      }
      if ((mask & 2) && act) {
        auto TB = [&](int c, int dy, int dx) -> double { return S2[c * PS + o + dy * W + dx]; };
        double aB[3];
        Th::accel(TB, p, Bz, aB);
#pragma unroll
        for (int c = 0; c < 3; ++c) A2[c * PO + s] = aB[c];
      }
    }
    __syncthreads();
    row_sums();
    // the next step's stage fields, assuming this step is not arrested (the common case): their
    // pushes travel under the same cluster barrier as the row sums
    const bool more = it + 1 < a.steps;
    if (more) P1(false);
    cluster.sync();

    // ---- P4: canonical y-tree, E, Q, KE, arrest (finalize_kernel), in every CTA
    y_tree();
    __syncthreads();
    if (wid < 3) {
      const double t = warp_tree(ysh[wid * 32 + lane]);
      if (lane == 0) tot[wid] = t;
    }
    __syncthreads();
    {
      const double E = a.h2 * tot[0], Q = a.h2 * tot[1], KE = a.h2 * tot[2];
      st.step += 1;
      const bool arrest = E > st.E_prev;  // strict; NaN compares false
      if (!isfinite(E)) st.nonfinite = 1;
      st.v_is_zero = arrest ? 1 : 0;
      if (arrest) {
        if (rank == 0 && tid == 0 && st.n_arrests < a.log_cap)
          a.log[(long long)b * a.log_cap + st.n_arrests] = st.step;
        st.n_arrests += 1;
      }
      st.E = E; st.Q = Q; st.KE = KE; st.E_prev = E;
      vz = arrest;
    }
    __syncthreads();  // tot is rewritten by the next step
    if (vz && more) {  // arrested (every CTA takes the same decision): redo the stage fields
      P1(true);
      cluster.sync();
    }
  }

  // ---- store the state
  for (int s = tid; s < nsite; s += RES_THREADS) {
    const int r = s / W, x = s - r * W, gy = gy0 + r;
    if (!active_site(x, gy)) continue;
    const long long o = (long long)gy * Nx + x;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      a.phi[lat + c * p.plane + o] = phi[c * PS + (r + 2) * W + x];
      a.vel[lat + c * p.plane + o] = vel[c * PO + s];
      a.a1[lat + c * p.plane + o] = A1[c * PO + s];
      a.a2[lat + c * p.plane + o] = A2[c * PO + s];
    }
  }
  if (rank == 0 && tid == 0) a.state[b] = st;
  cluster.sync();  // no CTA may exit while a neighbour still reads its shared memory
}

}  // namespace ss
