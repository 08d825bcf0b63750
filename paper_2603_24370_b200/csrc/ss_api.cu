// Host side of libss.so: the C ABI of include/ss.h.  Handle, workspace carving, the per-step
// CUDA graph (built with explicit kernel nodes so it can be replayed on any caller stream,
// including the legacy default stream), and the scalar read-outs.
#include "../../include/ss.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "ss_bs.cuh"
#include "ss_demag.cuh"
#include "ss_flow.cuh"
#include "ss_kernels.cuh"
#include "ss_render.cuh"
#include "ss_resident.cuh"

using namespace ss;

namespace {

thread_local char g_cuda_msg[256] = "";

inline bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA failure in %s: %s", what, cudaGetErrorString(e));
  return false;
}
#define CK(call)                                  \
  do {                                            \
    if (!cuda_ok((call), #call)) return SS_ERR_CUDA; \
  } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

constexpr int MULTI = 8;  // steps per multi-step graph (even)

struct MgHostLevel {
  size_t off_psi, off_tmp, off_rhs;  // [batch][ny+4][nx+4] fp64 each
  int nx, ny;
  double c;                          // 1 / (12 h_l^2)
};

struct Layout {
  size_t field_bytes;  // one [batch][C][Ny][Nx] array
  size_t part_bytes;   // one [batch][Ny][nseg] fp64 array
  size_t rows_bytes;   // [batch][3][Ny]
  size_t state_bytes, log_bytes, bb_bytes, render_bytes;
  int nacc;            // acceleration arrays: a1, a2 (+ a3 for the baby-Skyrme stage kernels)
  size_t off_phi[2], off_vel[2], off_a[4], off_part[3], off_rows, off_state, off_log, off_bb;
  size_t off_render;   // ss_render scratch: block extrema of one lattice, extrema, flag
  std::vector<MgHostLevel> mg;  // demagnetisation: multigrid hierarchy (level 0 = the lattice)
  size_t off_mg, mg_bytes;
  size_t total;
  int nseg;
};

// Limits of this build (include/ss.h "Limits"): the x-tree of row_reduce_kernel covers 32 lanes x
// 32 segment partials of 64 sites, the y-tree of finalize_kernel 1024 threads x 32 rows, and the
// lattice index is blockIdx.z.
constexpr int MAX_NX = 65536, MAX_NY = 32768, MAX_BATCH = 65535;
bool supported_shape(int Nx, int Ny, const ss_params* p) {
  return Nx <= MAX_NX && Ny <= MAX_NY && p->batch <= MAX_BATCH;
}

bool valid_shape(int theory, int Nx, int Ny, const ss_params* p) {
  if (!p) return false;
  if (theory != SS_THEORY_CHIRAL_MAGNET && theory != SS_THEORY_ABELIAN_HIGGS &&
      theory != SS_THEORY_BABY_SKYRME)
    return false;
  if (theory == SS_THEORY_BABY_SKYRME &&
      (p->potential < SS_POT_STANDARD || p->potential > SS_POT_BROKEN ||
       (p->potential == SS_POT_BROKEN && (p->potential_n < 1 || p->potential_n > 16))))
    return false;
  if (p->dtype != SS_F64 && p->dtype != SS_F32) return false;
  if (Nx < 5 || Ny < 5 || p->batch < 1) return false;
  if (p->dtype == SS_F64 ? (Nx % 2 != 0) : (Nx % 4 != 0)) return false;
  if (p->arrest_log_capacity < 0) return false;
  return true;
}

Layout make_layout(int theory, int Nx, int Ny, const ss_params* p) {
  Layout L;
  const int C = theory == SS_THEORY_ABELIAN_HIGGS ? 4 : 3;
  const size_t R = p->dtype == SS_F64 ? 8 : 4;
  L.nacc = theory == SS_THEORY_BABY_SKYRME ? 3 : 2;  // the per-stage schedule stores a3 as well
  if (theory == SS_THEORY_CHIRAL_MAGNET && p->demag != 0.0 && p->integrator == SS_RK4)
    L.nacc = 4;                                       // RK4 with one Poisson solve per stage
  const size_t cap = p->arrest_log_capacity > 0 ? (size_t)p->arrest_log_capacity : 4096;
  L.nseg = (Nx + SEG - 1) / SEG;
  L.field_bytes = align_up((size_t)p->batch * C * Ny * Nx * R);
  L.part_bytes = align_up((size_t)p->batch * Ny * L.nseg * sizeof(double));
  L.rows_bytes = align_up((size_t)p->batch * 3 * Ny * sizeof(double));
  L.state_bytes = align_up((size_t)p->batch * sizeof(LatticeState));
  L.log_bytes = align_up((size_t)p->batch * cap * sizeof(long long));
  L.bb_bytes = align_up((size_t)p->batch * sizeof(double));
  L.render_bytes = align_up((2 * (((size_t)Nx * Ny + 255) / 256) + 4) * sizeof(double));
  size_t o = 0;
  for (int i = 0; i < 2; ++i) { L.off_phi[i] = o; o += L.field_bytes; }
  for (int i = 0; i < 2; ++i) { L.off_vel[i] = o; o += L.field_bytes; }
  for (int i = 0; i < L.nacc; ++i) { L.off_a[i] = o; o += L.field_bytes; }
  for (int i = 0; i < 3; ++i) { L.off_part[i] = o; o += L.part_bytes; }
  L.off_rows = o; o += L.rows_bytes;
  L.off_state = o; o += L.state_bytes;
  L.off_log = o; o += L.log_bytes;
  L.off_bb = o; o += L.bb_bytes;
  L.off_render = o; o += L.render_bytes;
  L.off_mg = o; L.mg_bytes = 0;
  if (theory == SS_THEORY_CHIRAL_MAGNET && p->demag != 0.0) {
    int nx = Nx - 4, ny = Ny - 4;
    for (int l = 0;; ++l) {
      MgHostLevel lv;
      const size_t bytes = align_up((size_t)p->batch * (ny + 4) * (nx + 4) * sizeof(double));
      lv.nx = nx; lv.ny = ny;
      lv.c = 0.0;  // filled by ss_create (needs h)
      lv.off_psi = o; o += bytes;
      lv.off_tmp = o; o += bytes;
      lv.off_rhs = o; o += bytes;
      L.mg.push_back(lv);
      if ((nx <= MG_COARSE_MAX && ny <= MG_COARSE_MAX) || nx / 2 < 2 || ny / 2 < 2) break;
      nx /= 2; ny /= 2;
    }
    L.mg_bytes = o - L.off_mg;
  }
  L.total = o;
  return L;
}

struct KernelNode {
  void* func;
  dim3 grid, block;
  size_t smem;
  std::vector<unsigned char> args;  // the single by-value argument struct
  const char* name;
  std::vector<int> back;            // graph edges: waits for nodes i - back[k]; empty = {1}
};
inline void set_args(KernelNode& n, const void* a, size_t bytes) {
  n.args.resize(bytes);
  memcpy(n.args.data(), a, bytes);
}

}  // namespace

struct ss_solver {
  int theory, dtype, C, Nx, Ny, batch;
  int device, sms;  // the device the workspace lives on (current at ss_create) and its SM count
  double h, dt, kappa, B, K, lambda, mu, demag;
  int demag_cycles;
  int pot, potN;
  size_t R;
  cudaStream_t stream;
  char* ws;
  Layout L;
  long long log_cap;
  int flags;
  bool fields_set;
  int cur;  // which ping-pong buffer holds (phi, v)
  int cps[4];  // chunks per y-segment of flow kernels X, Y, V, XD
  int xkind;   // KX, or KXD (phi by TMA straight into ring A: fp64, not Abelian Higgs, no row slabs)
  int integrator;
  int ktheory;    // kernel family: kCM, kAH or kCMG (chiral magnet with a DMI table)
  double dmi[6];  // (d_x, d_y) of the table
  int64_t steps_done, launches;
  std::vector<KernelNode> step_nodes[2];  // per parity: Y, X (or V), row_reduce, finalize
  std::vector<KernelNode> prof_nodes[2];  // slab schedule: the unsplit Y, X, reductions (profiling)
  int slabs;                              // > 1: row-slab pipelined RK4 step
  std::vector<KernelNode> eval_nodes[2];  // X, row_reduce, finalize(advance = 0)
  cudaGraphExec_t step_exec[2];   // one flow step, per ping-pong parity
  cudaGraphExec_t multi_exec[2];  // MULTI consecutive steps in one graph (k steps per launch)
  std::vector<unsigned char> consts;  // FlowArgs<real> holding the per-site constants (ss_render)
  int res_cl, res_rows;               // resident-cluster schedule: cluster size (0 = off), rows/CTA
  size_t res_smem;
  std::vector<LatticeState> host_state;
  std::vector<double> Bb_host;  // per-lattice Zeeman field (host copy)

  void* phi(int i) const { return ws + L.off_phi[i]; }
  void* vel(int i) const { return ws + L.off_vel[i]; }
  void* acc(int i) const { return ws + L.off_a[i]; }
  double* part(int i) const { return (double*)(ws + L.off_part[i]); }
  LatticeState* state() const { return (LatticeState*)(ws + L.off_state); }
};

namespace {

// Every entry point runs on the solver's device whatever device is current in the calling thread
// (the kernels, graph launches and copies carry no device of their own) and restores the caller's.
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(const ss_solver* s) {
    if (!s) return;
    ok = cuda_ok(cudaGetDevice(&prev), "cudaGetDevice");
    if (ok && prev != s->device) ok = cuda_ok(cudaSetDevice(s->device), "cudaSetDevice");
    else prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define GUARD(s)            \
  DeviceGuard guard_(s);    \
  if (!guard_.ok) return SS_ERR_CUDA

// cuTensorMapEncodeTiled through the runtime (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) ==
            cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// field array [batch*C][Ny][Nx] as a 3-D tensor; box = {FW + 2*XPAD, FR, C} starting 16 bytes
// left of the strip (XPAD = 2 doubles / 4 floats); zero fill outside
bool make_tmap(const ss_solver* s, void* base, CUtensorMap* out, bool per_component = false) {
  EncodeTiledFn enc = encode_tiled();
  if (!enc) { snprintf(g_cuda_msg, sizeof(g_cuda_msg), "cuTensorMapEncodeTiled unavailable"); return false; }
  cuuint64_t dims[3] = {(cuuint64_t)s->Nx, (cuuint64_t)s->Ny, (cuuint64_t)s->batch * s->C};
  cuuint64_t strides[2] = {(cuuint64_t)s->Nx * s->R, (cuuint64_t)s->Nx * s->Ny * s->R};
  cuuint32_t box[3] = {(cuuint32_t)(FW + 32 / s->R), (cuuint32_t)FR,
                       (cuuint32_t)(per_component ? 1 : s->C)};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(out, s->dtype == SS_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64
                                           : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                   3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return false;
  }
  return true;
}

template <int THEORY, typename real>
void* flow_func_t(int kind) {
  if constexpr (sizeof(real) == 8 && THEORY != kAH)
    if (kind == KXD) return (void*)flow_kernel<THEORY, real, KXD>;
  return kind == KX   ? (void*)flow_kernel<THEORY, real, KX>
         : kind == KY ? (void*)flow_kernel<THEORY, real, KY>
                      : (void*)flow_kernel<THEORY, real, KV>;
}
void* flow_func(int theory, int dtype, int kind) {
  if (theory == kCMG)
    return dtype == SS_F64 ? flow_func_t<kCMG, double>(kind) : flow_func_t<kCMG, float>(kind);
  if (theory == SS_THEORY_CHIRAL_MAGNET)
    return dtype == SS_F64 ? flow_func_t<kCM, double>(kind) : flow_func_t<kCM, float>(kind);
  return dtype == SS_F64 ? flow_func_t<kAH, double>(kind) : flow_func_t<kAH, float>(kind);
}
template <int THEORY, typename real>
int flow_smem_t(int kind) {
  if constexpr (sizeof(real) == 8 && THEORY != kAH)
    if (kind == KXD) return FlowCfg<THEORY, real, KXD>::SMEM;
  return kind == KX   ? FlowCfg<THEORY, real, KX>::SMEM
         : kind == KY ? FlowCfg<THEORY, real, KY>::SMEM
                      : FlowCfg<THEORY, real, KV>::SMEM;
}
int flow_smem(int theory, int dtype, int kind) {
  if (theory == kCMG)
    return dtype == SS_F64 ? flow_smem_t<kCMG, double>(kind) : flow_smem_t<kCMG, float>(kind);
  if (theory == SS_THEORY_CHIRAL_MAGNET)
    return dtype == SS_F64 ? flow_smem_t<kCM, double>(kind) : flow_smem_t<kCM, float>(kind);
  return dtype == SS_F64 ? flow_smem_t<kAH, double>(kind) : flow_smem_t<kAH, float>(kind);
}

template <int THEORY, typename real>
int flow_threads_t(int kind) {
  if constexpr (sizeof(real) == 8 && THEORY != kAH)
    if (kind == KXD) return FlowCfg<THEORY, real, KXD>::THREADS;
  return kind == KX   ? FlowCfg<THEORY, real, KX>::THREADS
         : kind == KY ? FlowCfg<THEORY, real, KY>::THREADS
                      : FlowCfg<THEORY, real, KV>::THREADS;
}
int flow_threads(int theory, int dtype, int kind) {
  if (theory == kCMG)
    return dtype == SS_F64 ? flow_threads_t<kCMG, double>(kind) : flow_threads_t<kCMG, float>(kind);
  if (theory == SS_THEORY_CHIRAL_MAGNET)
    return dtype == SS_F64 ? flow_threads_t<kCM, double>(kind) : flow_threads_t<kCM, float>(kind);
  return dtype == SS_F64 ? flow_threads_t<kAH, double>(kind) : flow_threads_t<kAH, float>(kind);
}

// per-site constants: time-step combinations, folded stencil weights, theory parameters
template <typename real>
void fill_constants(const ss_solver* s, FlowArgs<real>& a) {
  const double dt = s->dt, h = s->h;
  a.Nx = s->Nx; a.Ny = s->Ny; a.nseg = s->L.nseg;
  a.plane = (long long)s->Nx * s->Ny;
  a.hdt = real(0.5 * dt); a.dt = real(dt);
  a.qdt2 = real(0.25 * (dt * dt)); a.hdt2 = real(0.5 * (dt * dt));
  a.sdt2 = real((dt * dt) / 6.0); a.sdt = real(dt / 6.0);
  a.i12h = real(1.0 / (12.0 * h)); a.i12h2 = real(1.0 / (12.0 * h * h));
  a.kappa = real(s->kappa); a.K = real(s->K); a.lambda = real(s->lambda);
  a.lap0 = real(60.0 / (12.0 * h * h)); a.lap1 = real(16.0 / (12.0 * h * h));
  a.lap2 = real(1.0 / (12.0 * h * h));
  a.dm1 = real(2.0 * s->kappa * 8.0 / (12.0 * h)); a.dm2 = real(2.0 * s->kappa / (12.0 * h));
  a.K2 = real(2.0 * s->K);
  a.jA = real((16.0 / 12.0) / (4.0 * h * h)); a.jB = real((-1.0 / 12.0) / (4.0 * h * h));
  a.hk = real(s->kappa / (12.0 * h));
  a.qs = real(1.0 / (4.0 * 3.14159265358979323846 * (12.0 * h) * (12.0 * h)));
  for (int i = 0; i < 6; ++i) a.dk[i] = real(s->kappa / (12.0 * h) * s->dmi[i]);
  a.bs_k2 = real(s->kappa * s->kappa); a.bs_mu2 = real(s->mu * s->mu);
  a.bs_pot = s->pot; a.bs_potN = s->potN;
}

// kernel X (kind KX) evaluates the state in buffer `in`; kernels Y and V advance `in` -> `in ^ 1`
// (V also a: acc(in) -> acc(in ^ 1))
template <typename real>
bool make_flow_node(const ss_solver* s, int kind, int in, KernelNode* out, int seg0, int nsegy) {
  FlowArgs<real> a;
  memset(&a, 0, sizeof(a));
  if (!make_tmap(s, s->phi(in), &a.tm[0]) || !make_tmap(s, s->vel(in), &a.tm[1]) ||
      !make_tmap(s, s->acc(kind == KV ? in : 0), &a.tm[2]) || !make_tmap(s, s->acc(1), &a.tm[3]))
    return false;
  if (kind == KXD && !make_tmap(s, s->phi(in), &a.tm[2], true)) return false;  // phi, one component per box
  if (kind == KX || kind == KXD) {
    a.out0 = (real*)s->acc(0); a.out1 = (real*)s->acc(1);
    a.part0 = s->part(0); a.part1 = s->part(1);
  } else if (kind == KV) {
    a.out0 = (real*)s->phi(in ^ 1); a.out1 = (real*)s->vel(in ^ 1); a.out2 = (real*)s->acc(in ^ 1);
    a.part0 = s->part(0); a.part1 = s->part(1); a.part2 = s->part(2);
  } else {
    a.out0 = (real*)s->phi(in ^ 1); a.out1 = (real*)s->vel(in ^ 1);
    a.part0 = s->part(2); a.part1 = nullptr;
  }
  a.state = s->state();
  a.Bb = (const double*)(s->ws + s->L.off_bb);
  fill_constants(s, a);
  a.cps = s->cps[kind];
  a.seg0 = seg0;  // this launch covers y-segments [seg0, seg0 + nsegy); nsegy = 0: all of them
  KernelNode n;
  n.func = flow_func(s->ktheory, s->dtype, kind);
  const int NC = (s->Ny + FR - 1) / FR;
  n.grid = dim3(s->L.nseg, nsegy > 0 ? nsegy : (NC + s->cps[kind] - 1) / s->cps[kind], s->batch);
  n.block = dim3(flow_threads(s->ktheory, s->dtype, kind), 1, 1);
  n.smem = (size_t)flow_smem(s->ktheory, s->dtype, kind);
  set_args(n, &a, sizeof(a));
  n.name = (kind == KX || kind == KXD) ? "flow_x_grad_energy_charge_stage2"
           : kind == KY ? "flow_y_stage34_combine_project_ke"
                        : "flow_v_verlet_step_energy_charge_ke";
  *out = n;
  return true;
}
bool make_flow_node(const ss_solver* s, int kind, int in, KernelNode* out, int seg0 = 0, int nsegy = 0) {
  return s->dtype == SS_F64 ? make_flow_node<double>(s, kind, in, out, seg0, nsegy)
                            : make_flow_node<float>(s, kind, in, out, seg0, nsegy);
}

// baby Skyrme: one tile kernel per RK4 stage (ss_bs.cuh); stage 1 evaluates buffer `cur`,
// stages 2-4 advance `cur` -> `cur ^ 1`
template <typename real>
void* bs_func(int stage) {
  switch (stage) {
    case 1: return (void*)bs_stage_kernel<real, 1>;
    case 2: return (void*)bs_stage_kernel<real, 2>;
    case 3: return (void*)bs_stage_kernel<real, 3>;
    case 4: return (void*)bs_stage_kernel<real, 4>;
    default: return (void*)bs_stage_kernel<real, 5>;
  }
}
template <typename real>
KernelNode make_bs_node(const ss_solver* s, int stage, int cur) {
  FlowArgs<real> k;
  memset(&k, 0, sizeof(k));
  fill_constants(s, k);
  BsArgs<real> a;
  memset(&a, 0, sizeof(a));
  a.phi = (const real*)s->phi(cur);
  a.vel = (const real*)s->vel(cur);
  a.aprev = stage == 3 ? (const real*)s->acc(0) : (const real*)s->acc(1);  // stage 4: a2
  a.aout = (real*)s->acc(stage == 1 ? 0 : stage == 2 ? 1 : 2);
  if (s->integrator == SS_VERLET) {  // stage 5 steps cur -> cur ^ 1; stage 1 evaluates buffer cur
    a.aprev = (const real*)s->acc(cur);
    a.aout = (real*)s->acc(stage == 1 ? cur : cur ^ 1);
  }
  a.a1 = (const real*)s->acc(0);
  a.a3 = (const real*)s->acc(2);
  a.phi_out = (real*)s->phi(cur ^ 1);
  a.vel_out = (real*)s->vel(cur ^ 1);
  a.part_e = s->part(0); a.part_q = s->part(1); a.part_ke = s->part(2);
  a.state = s->state();
  a.Nx = s->Nx; a.Ny = s->Ny; a.nseg = s->L.nseg; a.plane = k.plane;
  // stage fields: phi2 = R(phi + dt/2 v), phi3 = R((phi + dt/2 v) + dt^2/4 a1),
  // phi4 = R((phi + dt v) + dt^2/2 a2)
  a.alpha = stage == 4 ? k.dt : k.hdt;
  a.beta = stage == 5 ? k.hdt : (stage == 3 ? k.qdt2 : k.hdt2);
  a.dt = k.dt; a.sdt2 = k.sdt2; a.sdt = k.sdt;
  a.i12h = k.i12h; a.i12h2 = k.i12h2;
  a.lap0 = k.lap0; a.lap1 = k.lap1; a.lap2 = k.lap2;
  a.jA = k.jA; a.jB = k.jB;
  a.bs_k2 = k.bs_k2; a.bs_mu2 = k.bs_mu2; a.bs_pot = k.bs_pot; a.bs_potN = k.bs_potN;
  KernelNode n;
  n.func = bs_func<real>(stage);
  n.grid = dim3((s->Nx + BTX - 1) / BTX, (s->Ny + BTY - 1) / BTY, s->batch);
  n.block = dim3(BBX, BBY, 1);
  n.smem = sizeof(BsSmem<real>);
  set_args(n, &a, sizeof(a));
  static const char* names[5] = {"bs_stage1_grad_energy_charge", "bs_stage2", "bs_stage3",
                                 "bs_stage4_combine_project_ke", "bs_verlet_step_energy_charge_ke"};
  n.name = names[stage - 1];
  return n;
}
KernelNode make_bs_node(const ss_solver* s, int stage, int cur) {
  return s->dtype == SS_F64 ? make_bs_node<double>(s, stage, cur)
                            : make_bs_node<float>(s, stage, cur);
}

// ---- demagnetisation (ss_demag.cuh): nodes of n V-cycles and of the Verlet step around them
KernelNode mg_node(void* func, const MgArgs& m, dim3 grid, dim3 block, size_t smem, const char* name) {
  KernelNode n;
  n.func = func; n.grid = grid; n.block = block; n.smem = smem; n.name = name;
  set_args(n, &m, sizeof(m));
  return n;
}
void add_vcycle(const ss_solver* s, size_t l, std::vector<KernelNode>& out) {
  const MgHostLevel& f = s->L.mg[l];
  double* psi = (double*)(s->ws + f.off_psi);
  double* tmp = (double*)(s->ws + f.off_tmp);
  const double* rhs = (const double*)(s->ws + f.off_rhs);
  const dim3 block(MGX, MGY, 1);
  const dim3 grid((f.nx + MGX - 1) / MGX, (f.ny + MGY - 1) / MGY, s->batch);
  MgArgs m;
  memset(&m, 0, sizeof(m));
  m.nx = f.nx; m.ny = f.ny; m.c = f.c; m.rhs = rhs;
  if (l > 0) {  // wall images: psi(-k) = (d - k)/d psi(0), d = distance of the wall-adjacent unknown
    m.walls = 1;   // from the physical wall in spacings of this level (ss_demag.cuh mg_store)
    const double sp = double(1 << l);
    const double dl = 0.5 + 0.5 / sp;  // unknown I of level l sits at 2^l I + (2^l - 1)/2 fine cells
    const double n0[2] = {double(s->L.mg[0].nx), double(s->L.mg[0].ny)};
    const int nl[2] = {f.nx, f.ny};
    for (int dim = 0; dim < 2; ++dim) {
      const double dr = (n0[dim] - (sp * (nl[dim] - 1) + (sp - 1.0) / 2.0)) / sp;
      for (int k = 1; k <= 2; ++k) {
        m.bw[4 * dim + k - 1] = (dl - k) / dl;
        m.bw[4 * dim + 2 + k - 1] = (dr - k) / dr;
      }
    }
  }
  if (l + 1 == s->L.mg.size()) {
    m.out = psi;
    out.push_back(mg_node((void*)mg_coarse_kernel, m, dim3(s->batch, 1, 1), dim3(1024, 1, 1),
                          (size_t)3 * (f.nx + 4) * (f.ny + 4) * sizeof(double), "mg_coarse"));
    return;
  }
  auto smooth2 = [&]() {  // two sweeps: psi -> tmp -> psi
    MgArgs a = m;
    a.in = psi; a.out = tmp;
    out.push_back(mg_node((void*)mg_smooth_kernel, a, grid, block, 0, "mg_smooth"));
    a.in = tmp; a.out = psi;
    out.push_back(mg_node((void*)mg_smooth_kernel, a, grid, block, 0, "mg_smooth"));
  };
  smooth2();
  const MgHostLevel& c = s->L.mg[l + 1];
  const dim3 cgrid((c.nx + MGX - 1) / MGX, (c.ny + MGY - 1) / MGY, s->batch);
  MgArgs r = m;
  r.in = psi; r.out = (double*)(s->ws + c.off_rhs); r.out2 = (double*)(s->ws + c.off_psi);
  r.cnx = c.nx; r.cny = c.ny;
  out.push_back(mg_node((void*)mg_restrict_kernel, r, cgrid, block, 0, "mg_residual_restrict"));
  add_vcycle(s, l + 1, out);
  MgArgs pr = m;
  pr.out = psi; pr.in = (const double*)(s->ws + c.off_psi); pr.cnx = c.nx; pr.cny = c.ny;
  out.push_back(mg_node((void*)mg_prolong_kernel, pr, grid, block, 0, "mg_prolong_add"));
  smooth2();
}
// step: drift(cur -> cur^1), rho, V-cycles, kick; evaluation (ss_set_fields): rho, 4x the V-cycles
// from psi = 0, kick without the velocity update
void make_demag_step(const ss_solver* s, int cur, std::vector<KernelNode>& st,
                     std::vector<KernelNode>& ev) {
  DemagStepArgs a;
  memset(&a, 0, sizeof(a));
  a.p = *reinterpret_cast<const FlowArgs<double>*>(s->consts.data());
  const MgHostLevel& l0 = s->L.mg[0];
  a.d.rho = (double*)(s->ws + l0.off_rhs);
  a.d.psi = (const double*)(s->ws + l0.off_psi);
  a.d.part_e = s->part(0); a.d.part_q = s->part(1); a.d.part_ke = s->part(2);
  a.d.state = s->state();
  a.d.Bb = (const double*)(s->ws + s->L.off_bb);
  a.d.g = s->demag;
  const long long plane = (long long)s->Nx * s->Ny;
  const dim3 pgrid((unsigned)((plane + 255) / 256), 1, s->batch);
  const dim3 kgrid((s->Nx + DTX - 1) / DTX, (s->Ny + DTY - 1) / DTY, s->batch);
  void* kick = s->ktheory == kCMG ? (void*)demag_kick_kernel<kCMG> : (void*)demag_kick_kernel<kCM>;
  auto node = [&](void* f, const DemagStepArgs& x, dim3 grid, dim3 block, const char* name) {
    KernelNode n;
    n.func = f; n.grid = grid; n.block = block; n.smem = 0; n.name = name;
    set_args(n, &x, sizeof(x));
    return n;
  };
  if (s->integrator == SS_RK4) {  // one Poisson solve per stage field (ss_demag.cuh header)
    const FlowArgs<double>& k = a.p;
    double* S = (double*)s->phi(cur ^ 1);  // stage fields live where phi' goes at the end
    for (int stage = 2; stage <= 4; ++stage) {
      DemagStepArgs x = a;
      x.d.phi = (const double*)s->phi(cur); x.d.vel = (const double*)s->vel(cur);
      x.d.acc = stage == 3 ? (const double*)s->acc(0) : (const double*)s->acc(1);
      x.d.use_acc = stage > 2;
      x.d.alpha = stage == 4 ? k.dt : k.hdt;
      x.d.beta = stage == 3 ? k.qdt2 : k.hdt2;
      x.d.phi_out = S;
      st.push_back(node((void*)demag_stage_kernel, x, pgrid, dim3(256, 1, 1), "demag_stage_field"));
      x.d.phi = S;
      st.push_back(node((void*)demag_rho_kernel, x, pgrid, dim3(256, 1, 1), "demag_rho"));
      for (int c = 0; c < s->demag_cycles; ++c) add_vcycle(s, 0, st);
      x.d.acc_out = (double*)s->acc(stage - 1);
      x.d.advance = 2;
      st.push_back(node(kick, x, kgrid, dim3(DBX, DBY, 1), "demag_stage_accel"));
    }
    DemagStepArgs x = a;
    x.d.phi = (const double*)s->phi(cur); x.d.vel = (const double*)s->vel(cur);
    x.d.a1 = (const double*)s->acc(0); x.d.a2 = (const double*)s->acc(1);
    x.d.a3 = (const double*)s->acc(2); x.d.a4 = (const double*)s->acc(3);
    x.d.phi_out = (double*)s->phi(cur ^ 1); x.d.vel_out = (double*)s->vel(cur ^ 1);
    st.push_back(node((void*)demag_combine_kernel, x, kgrid, dim3(DBX, DBY, 1),
                      "demag_rk4_combine_project_ke"));
    x.d.phi = (const double*)s->phi(cur ^ 1);
    st.push_back(node((void*)demag_rho_kernel, x, pgrid, dim3(256, 1, 1), "demag_rho"));
    for (int c = 0; c < s->demag_cycles; ++c) add_vcycle(s, 0, st);
    x.d.acc_out = (double*)s->acc(0);
    x.d.advance = 0;
    st.push_back(node(kick, x, kgrid, dim3(DBX, DBY, 1), "demag_kick_energy_charge_ke"));
  } else {  // one Verlet step
    DemagStepArgs x = a;
    x.d.phi = (const double*)s->phi(cur); x.d.vel = (const double*)s->vel(cur);
    x.d.acc = (const double*)s->acc(cur);
    x.d.phi_out = (double*)s->phi(cur ^ 1); x.d.vel_out = (double*)s->vel(cur ^ 1);
    st.push_back(node((void*)demag_drift_kernel, x, pgrid, dim3(256, 1, 1), "demag_drift"));
    x.d.phi = (const double*)s->phi(cur ^ 1);
    st.push_back(node((void*)demag_rho_kernel, x, pgrid, dim3(256, 1, 1), "demag_rho"));
    for (int c = 0; c < s->demag_cycles; ++c) add_vcycle(s, 0, st);
    x.d.vel = (const double*)s->vel(cur ^ 1); x.d.vel_out = (double*)s->vel(cur ^ 1);
    x.d.acc_out = (double*)s->acc(cur ^ 1);
    x.d.advance = 1;
    st.push_back(node(kick, x, kgrid, dim3(DBX, DBY, 1), "demag_kick_energy_charge_ke"));
  }
  {  // evaluation of the state in buffer cur (only used with cur == 0)
    DemagStepArgs x = a;
    x.d.phi = (const double*)s->phi(cur);
    ev.push_back(node((void*)demag_rho_kernel, x, pgrid, dim3(256, 1, 1), "demag_rho"));
    for (int c = 0; c < 4 * s->demag_cycles; ++c) add_vcycle(s, 0, ev);
    x.d.acc_out = (double*)s->acc(s->integrator == SS_RK4 ? 0 : cur);
    x.d.advance = 0;
    ev.push_back(node(kick, x, kgrid, dim3(DBX, DBY, 1), "demag_kick_energy_charge_ke"));
  }
}

// chunks per segment: minimise (waves of CTAs) x (chunks marched per CTA, warm-up included)
int choose_cps(int nstrips, int Ny, int batch, int slots) {
  const int NC = (Ny + FR - 1) / FR;
  long long best = -1;
  int best_cps = 1;
  for (int cps = 1; cps <= NC; ++cps) {
    const long long items = (long long)nstrips * ((NC + cps - 1) / cps) * batch;
    const long long waves = (items + slots - 1) / slots;
    const long long cost = waves * (4 * (cps + 2) + 3);  // + per-CTA prologue
    if (best < 0 || cost < best) { best = cost; best_cps = cps; }
  }
  return best_cps;
}

// Row-slab pipelining of the RK4 step (ss_create): lattices tall enough for SLABS slabs of at
// least two segments each, and at least two waves of CTAs -- below that the split only costs
// (cm 1024^2: 0.084 vs 0.074 ms, 1280^2: 0.107 vs 0.109).  Batched lattices are split the same
// way, every slab launch covering its rows of all lattices (4 x 1024^2: 0.246 -> 0.227 ms, 16 x
// 512^2: 0.283 -> 0.237, 2 x 2048^2: 0.459 -> 0.406); many small lattices do not qualify (256 x
// 256^2: two segments of four waves' length per lattice; split by lattice instead: -0.3 %, not
// built).  With the tail of Y filled by X the best segment is shorter than
// choose_cps's: about four waves of CTAs in all, not below 8 chunks (measured: cm 4096^2 fp64
// flat over 22..38 chunks, fp32 best at 24, Abelian Higgs 2048^2 best at 14..16, cm 1536^2 and
// 1792^2 best at 8: 0.139 vs 0.146 and 0.178 vs 0.192 ms without slabs).
constexpr int SLABS = 4;
void plan_slabs(ss_solver* s, int user_cps, int slots) {
  s->slabs = 0;
  if (s->integrator != SS_RK4 || s->ktheory == kBS || s->demag != 0.0) return;
  const int min_nsy = s->batch > 1 ? SLABS : 2 * SLABS;
  if (s->flags & SS_FLAG_NO_SLABS) return;
  const int NC = (s->Ny + FR - 1) / FR;
  int cps = user_cps;
  if (cps <= 0) {
    const int segs = (4 * slots + s->L.nseg * s->batch - 1) / (s->L.nseg * s->batch);
    cps = (NC + segs - 1) / (segs > 0 ? segs : 1);
    if (cps < 8) cps = 8;
    // many lattices: the formula above leaves fewer than eight segments per lattice; one segment
    // per slab of at least 16 chunks still pays (256 x 256^2: 0.922 -> 0.904 ms, 64 x 512^2: 1.00
    // -> 0.84, 16 x 1024^2: 0.849 -> 0.807)
    if (s->batch > 1 && (NC + cps - 1) / cps < 2 * SLABS) cps = std::max(16, (NC + 2 * SLABS - 1) / (2 * SLABS));
  }
  const int nsy = (NC + cps - 1) / cps;
  if (nsy < min_nsy || (long long)nsy * s->L.nseg * s->batch < 2LL * slots) return;
  s->slabs = SLABS;
  s->cps[KX] = s->cps[KY] = cps;
}

// row_reduce of rows [row0, row1) alone (the slab schedule finishes the rows of a slab as soon as
// its X is done)
KernelNode make_row_reduce_node(const ss_solver* s, int row0, int row1);
void make_reduce_nodes(const ss_solver* s, int advance, std::vector<KernelNode>& out,
                       bool finalize_only = false) {
  ReduceArgs a;
  memset(&a, 0, sizeof(a));
  a.part_e = s->part(0);
  a.part_q = s->part(1);
  a.part_ke = s->part(2);
  a.rows = (double*)(s->ws + s->L.off_rows);
  a.state = s->state();
  a.log = (long long*)(s->ws + s->L.off_log);
  a.log_cap = s->log_cap;
  a.Ny = s->Ny; a.nseg = s->L.nseg; a.advance = advance;
  a.h2 = s->h * s->h;
  a.row0 = 0; a.row1 = s->Ny;
  KernelNode r;
  r.func = (void*)row_reduce_kernel;
  r.grid = dim3((s->Ny + 7) / 8, s->batch, 1);
  r.block = dim3(256, 1, 1);
  r.smem = 0;
  set_args(r, &a, sizeof(a));
  r.name = "row_reduce";
  if (!finalize_only) out.push_back(r);
  KernelNode f = r;
  f.name = "finalize_arrest";
  f.func = (void*)finalize_kernel;
  f.grid = dim3(s->batch, 1, 1);
  f.block = dim3(1024, 1, 1);
  out.push_back(f);
}

KernelNode make_row_reduce_node(const ss_solver* s, int row0, int row1) {
  std::vector<KernelNode> both;
  make_reduce_nodes(s, 1, both);
  KernelNode r = both[0];
  ReduceArgs a;
  memcpy(&a, r.args.data(), sizeof(a));
  a.row0 = row0; a.row1 = row1;
  set_args(r, &a, sizeof(a));
  r.grid = dim3((row1 - row0 + 7) / 8, s->batch, 1);
  return r;
}

int launch_nodes(ss_solver* s, std::vector<KernelNode>& nodes) {
  for (auto& n : nodes) {
    void* params[1] = {n.args.data()};
    CK(cudaLaunchKernel(n.func, n.grid, n.block, params, n.smem, s->stream));
    s->launches += 1;
  }
  return SS_OK;
}

int build_graph(ss_solver* s, std::vector<KernelNode>& nodes, cudaGraphExec_t* exec) {
  cudaGraph_t g;
  CK(cudaGraphCreate(&g, 0));
  std::vector<cudaGraphNode_t> made;
  for (auto& n : nodes) {
    cudaKernelNodeParams kp;
    memset(&kp, 0, sizeof(kp));
    void* params[1] = {n.args.data()};
    kp.func = n.func;
    kp.gridDim = n.grid;
    kp.blockDim = n.block;
    kp.sharedMemBytes = (unsigned)n.smem;
    kp.kernelParams = params;
    cudaGraphNode_t node;
    std::vector<cudaGraphNode_t> deps;
    const int i = (int)made.size();
    if (n.back.empty()) {
      if (i > 0) deps.push_back(made[i - 1]);
    } else {
      for (int bk : n.back)
        if (i - bk >= 0) deps.push_back(made[i - bk]);
    }
    cudaError_t e = cudaGraphAddKernelNode(&node, g, deps.data(), deps.size(), &kp);
    if (!cuda_ok(e, "cudaGraphAddKernelNode")) { cudaGraphDestroy(g); return SS_ERR_CUDA; }
    made.push_back(node);
  }
  cudaError_t e = cudaGraphInstantiate(exec, g, 0);
  cudaGraphDestroy(g);
  if (!cuda_ok(e, "cudaGraphInstantiate")) return SS_ERR_CUDA;
  // upload now: otherwise the first launch of each graph pays for it inside the caller's timing
  if (!cuda_ok(cudaGraphUpload(*exec, s->stream), "cudaGraphUpload")) return SS_ERR_CUDA;
  return SS_OK;
}

// Resident-cluster schedule (ss_resident.cuh): chiral magnet, default DMI, fp64, RK4, lattices
// whose state fits in the shared memory of one cluster and whose clusters fit on the device at once
void choose_resident(ss_solver* s) {
  s->res_cl = 0;
  if (s->ktheory != kCM || s->dtype != SS_F64 || s->integrator != SS_RK4 || s->demag != 0.0) return;
  if (s->flags & SS_FLAG_NO_RESIDENT) return;
  if (s->Nx % 32 != 0 || s->Nx > 1024 || s->Ny > RES_MAX_NY) return;
  const int order[5] = {16, 8, 4, 2, 1};  // most SMs first: the fp64 pipes bound the step
  for (int i = 0; i < 5; ++i) {
    const int cl = order[i];
    if (s->Ny % cl != 0 || (cl > 1 && s->Ny / cl < 2 * HALO)) continue;
    if ((long long)cl * s->batch > s->sms) continue;
    const size_t smem = resident_smem_doubles(s->Nx, s->Ny, s->Ny / cl) * sizeof(double);
    if (smem > 227 * 1024) continue;
    if (cudaFuncSetAttribute((void*)resident_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)smem) != cudaSuccess ||
        (cl > 8 && cudaFuncSetAttribute((void*)resident_kernel,
                                        cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess)) {
      cudaGetLastError();
      continue;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(cl, s->batch, 1);
    cfg.blockDim = dim3(RES_THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, (void*)resident_kernel, &cfg) != cudaSuccess ||
        nclusters < s->batch) {
      cudaGetLastError();
      continue;
    }
    s->res_cl = cl; s->res_rows = s->Ny / cl; s->res_smem = smem;
    return;
  }
}

int resident_step(ss_solver* s, int64_t k) {
  ResidentArgs a;
  memset(&a, 0, sizeof(a));
  a.k = *reinterpret_cast<const FlowArgs<double>*>(s->consts.data());
  a.phi = (double*)s->phi(s->cur); a.vel = (double*)s->vel(s->cur);
  a.a1 = (double*)s->acc(0); a.a2 = (double*)s->acc(1);
  a.state = s->state();
  a.log = (long long*)(s->ws + s->L.off_log);
  a.log_cap = s->log_cap;
  a.Bb = (const double*)(s->ws + s->L.off_bb);
  a.rows = s->res_rows;
  a.steps = k;
  a.h2 = s->h * s->h;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(s->res_cl, s->batch, 1);
  cfg.blockDim = dim3(RES_THREADS, 1, 1);
  cfg.dynamicSmemBytes = s->res_smem;
  cfg.stream = s->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = s->res_cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  CK(cudaLaunchKernelEx(&cfg, resident_kernel, a));
  s->launches += 1;
  s->steps_done += k;
  return SS_OK;
}

int read_state(ss_solver* s) {
  CK(cudaMemcpyAsync(s->host_state.data(), s->state(), s->batch * sizeof(LatticeState),
                     cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return SS_OK;
}

}  // namespace

extern "C" {

size_t ss_workspace_bytes(int theory, int Nx, int Ny, const ss_params* p) {
  if (!valid_shape(theory, Nx, Ny, p) || !supported_shape(Nx, Ny, p)) return 0;
  return make_layout(theory, Nx, Ny, p).total;
}

int ss_create(ss_solver** out, int theory, int Nx, int Ny, double h, const ss_params* p) {
  if (!out) return SS_ERR_ARG;
  *out = nullptr;
  if (!valid_shape(theory, Nx, Ny, p) || !(h > 0.0) || !std::isfinite(h)) return SS_ERR_ARG;
  if (p->integrator != SS_RK4 && p->integrator != SS_VERLET) return SS_ERR_ARG;
  if (p->flags & ~(SS_FLAG_NO_GRAPH | SS_FLAG_NO_RESIDENT | SS_FLAG_NO_SLABS)) return SS_ERR_ARG;
  if (theory == SS_THEORY_BABY_SKYRME && p->dmi_d) return SS_ERR_UNSUPPORTED;
  if (!std::isfinite(p->demag) || p->demag < 0.0 || p->demag_cycles < 0) return SS_ERR_ARG;
  if (p->demag != 0.0 && theory == SS_THEORY_CHIRAL_MAGNET && p->dtype != SS_F64)
    return SS_ERR_UNSUPPORTED;  // demagnetisation: fp64 only
  if (p->dmi_d)
    for (int i = 0; i < 6; ++i)
      if (!std::isfinite(p->dmi_d[i])) return SS_ERR_ARG;
  if (!supported_shape(Nx, Ny, p)) return SS_ERR_UNSUPPORTED;
  int ndev = 0;
  if (!cuda_ok(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount") || ndev == 0) {
    if (ndev == 0) snprintf(g_cuda_msg, sizeof(g_cuda_msg), "no CUDA device (libss has no CPU path)");
    return SS_ERR_CUDA;
  }
  Layout L = make_layout(theory, Nx, Ny, p);
  if (!p->workspace || p->workspace_bytes < L.total || ((uintptr_t)p->workspace & 255) != 0)
    return SS_ERR_WORKSPACE;
  cudaPointerAttributes pa;
  if (!cuda_ok(cudaPointerGetAttributes(&pa, p->workspace), "cudaPointerGetAttributes"))
    return SS_ERR_CUDA;
  if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return SS_ERR_WORKSPACE;
  ss_solver* s = new (std::nothrow) ss_solver();
  if (!s) return SS_ERR_ARG;
  s->theory = theory; s->dtype = p->dtype; s->C = theory == SS_THEORY_ABELIAN_HIGGS ? 4 : 3;
  s->mu = p->mu; s->pot = p->potential; s->potN = p->potential_n;
  s->demag = theory == SS_THEORY_CHIRAL_MAGNET ? p->demag : 0.0;
  s->demag_cycles = p->demag_cycles > 0 ? p->demag_cycles : 8;
  s->Nx = Nx; s->Ny = Ny; s->batch = p->batch; s->h = h;
  s->device = pa.device;
  s->dt = p->dt > 0.0 ? p->dt : 0.5 * h;
  s->kappa = p->kappa; s->B = p->B; s->K = p->K; s->lambda = p->lambda;
  s->R = p->dtype == SS_F64 ? 8 : 4;
  s->stream = (cudaStream_t)p->stream;
  s->ws = (char*)p->workspace;
  s->L = L;
  for (size_t l = 0; l < s->L.mg.size(); ++l) {
    const double hl = h * double(1 << l);
    s->L.mg[l].c = 1.0 / (12.0 * hl * hl);
  }
  if (s->demag != 0.0) {  // the coarsest level is relaxed by one CTA in shared memory
    const MgHostLevel& lv = s->L.mg.back();
    if ((size_t)3 * (lv.nx + 4) * (lv.ny + 4) * sizeof(double) > 200 * 1024) {
      delete s;
      return SS_ERR_UNSUPPORTED;  // very anisotropic lattice: no semi-coarsening in this build
    }
  }
  s->log_cap = p->arrest_log_capacity > 0 ? p->arrest_log_capacity : 4096;
  s->flags = p->flags;
  s->integrator = p->integrator;
  s->ktheory = theory == SS_THEORY_BABY_SKYRME ? kBS : theory;
  for (int i = 0; i < 6; ++i) s->dmi[i] = 0.0;
  if (theory == SS_THEORY_CHIRAL_MAGNET && p->dmi_d) {
    s->ktheory = kCMG;
    for (int i = 0; i < 6; ++i) s->dmi[i] = p->dmi_d[i];
  }
  s->fields_set = false;
  s->cur = 0;
  s->steps_done = 0; s->launches = 0;
  s->step_exec[0] = s->step_exec[1] = nullptr;
  s->multi_exec[0] = s->multi_exec[1] = nullptr;
  s->host_state.resize(s->batch);
  DeviceGuard guard(s);
  if (!guard.ok) { delete s; return SS_ERR_CUDA; }
  s->sms = 0;
  cudaError_t e = cudaDeviceGetAttribute(&s->sms, cudaDevAttrMultiProcessorCount, s->device);
  if (!cuda_ok(e, "cudaDeviceGetAttribute") || s->sms < 1) { delete s; return SS_ERR_CUDA; }

  std::vector<double> bb(s->batch, p->B);
  if (p->B_batch) bb.assign(p->B_batch, p->B_batch + s->batch);
  s->Bb_host = bb;
  e = cudaMemcpyAsync(s->ws + L.off_bb, bb.data(), s->batch * sizeof(double),
                      cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);  // bb is a local
  if (!cuda_ok(e, "upload B_batch")) { delete s; return SS_ERR_CUDA; }

  if (p->dtype == SS_F64) {
    FlowArgs<double> k;
    memset(&k, 0, sizeof(k));
    fill_constants(s, k);
    s->consts.assign((unsigned char*)&k, (unsigned char*)&k + sizeof(k));
  } else {
    FlowArgs<float> k;
    memset(&k, 0, sizeof(k));
    fill_constants(s, k);
    s->consts.assign((unsigned char*)&k, (unsigned char*)&k + sizeof(k));
  }
  if (s->demag != 0.0) {
    e = cudaFuncSetAttribute((void*)mg_coarse_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             200 * 1024);
    if (!cuda_ok(e, "cudaFuncSetAttribute")) { delete s; return SS_ERR_CUDA; }
  }
  if (s->ktheory == kBS) {
    for (int stage = 1; stage <= 5; ++stage) {
      void* f = p->dtype == SS_F64 ? bs_func<double>(stage) : bs_func<float>(stage);
      const size_t smem = p->dtype == SS_F64 ? sizeof(BsSmem<double>) : sizeof(BsSmem<float>);
      e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (!cuda_ok(e, "cudaFuncSetAttribute")) { delete s; return SS_ERR_CUDA; }
    }
  }
  int slots[3] = {1, 1, 1};
  const bool has_xd = p->dtype == SS_F64 && s->ktheory != kAH && s->ktheory != kBS;
  s->cps[KXD] = 1;
  for (int kind = 0; kind < (has_xd ? 4 : 3) && s->ktheory != kBS; ++kind) {
    void* f = flow_func(s->ktheory, p->dtype, kind);
    const int smem = flow_smem(s->ktheory, p->dtype, kind);
    e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (!cuda_ok(e, "cudaFuncSetAttribute")) { delete s; return SS_ERR_CUDA; }
    int o = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, f, flow_threads(s->ktheory, p->dtype, kind), smem);
    if (!cuda_ok(e, "cudaOccupancyMaxActiveBlocksPerMultiprocessor") || o < 1) {
      delete s; return SS_ERR_CUDA;
    }
    s->cps[kind] = p->chunks_per_segment > 0 ? p->chunks_per_segment
                                             : choose_cps(L.nseg, Ny, s->batch, s->sms * o);
    if (kind < 3) slots[kind] = s->sms * o;
  }
  plan_slabs(s, p->chunks_per_segment, slots[KX] < slots[KY] ? slots[KX] : slots[KY]);
  // Without row slabs kernel X takes phi by TMA straight into its ring (ss_flow.cuh KXD: 4 CTAs
  // per SM; 256 x 256^2 0.917 vs 0.936 ms, cm 512^2 ... 1536^2 and 4 ... 64 batched lattices 1 ... 8 %
  // faster than KX).  Inside the slab schedule
  // its single TMA stage waits longer while Y streams (cm 4096^2 0.807 vs 0.793): KX there.
  s->xkind = (has_xd && s->slabs == 0 && s->integrator == SS_RK4) ? KXD : KX;
  for (int cur = 0; cur < 2; ++cur) {
    auto& st = s->step_nodes[cur];
    auto& ev = s->eval_nodes[cur];
    int join = 1;  // > 1: slab schedule with that many slabs
    if (s->demag != 0.0) {
      make_demag_step(s, cur, st, ev);
    } else if (s->ktheory == kBS) {
      if (s->integrator == SS_VERLET) {
        st.push_back(make_bs_node(s, 5, cur));  // the whole step: phi', v', a', E, Q, KE
      } else {
        // stage 2 (phi, v -> a2) and stage 3 (phi, v, a1 -> a3) do not depend on one another:
        // both wait for the previous step's finalize only and share the device
        st.push_back(make_bs_node(s, 2, cur));
        st.push_back(make_bs_node(s, 3, cur));
        st.back().back = {2};
        st.push_back(make_bs_node(s, 4, cur));
        st.back().back = {1, 2};
        st.push_back(make_bs_node(s, 1, cur ^ 1));  // a1, E, Q on the new field
      }
      ev.push_back(make_bs_node(s, 1, cur));
    } else if (s->integrator == SS_VERLET) {
      KernelNode v, x0;
      if (!make_flow_node(s, KV, cur, &v) || !make_flow_node(s, KX, cur, &x0)) {
        ss_destroy(s);
        return SS_ERR_CUDA;
      }
      st.push_back(v);   // the whole step: phi', v', a', E, Q, KE
      ev.push_back(x0);  // a (-> acc(0), only used with cur == 0), E, Q
    } else if (s->slabs > 1) {
      // Row-slab pipelining (DESIGN 6.1): Y and X of one step as SLABS launches each over
      // contiguous ranges of y-segments.  X_k reads rows that Y_{k-1}, Y_k, Y_{k+1} write (one
      // chunk beyond its slab on either side) and overwrites a1, a2 rows that the same three
      // read, so those are its only edges; the Y_k depend on the previous step's arrest flag
      // alone.  X's CTAs fill the SMs that the tail of Y leaves idle, and the rows of a slab are
      // reduced (R_k) as soon as X_k is done, so that only the last slab's row_reduce and the
      // finalize are serial (0.7931 vs 0.7949 ms with one row_reduce at the end).  Node order (also
      // the order of the direct-launch path) is Y0 Y1 X0 R0 Y2 X1 R1 ...: topological.
      const int S = s->slabs;
      const int NC = (s->Ny + FR - 1) / FR;
      const int nsy = (NC + s->cps[KY] - 1) / s->cps[KY];
      std::vector<int> lo(S + 1), iy(S), ix(S);
      for (int k = 0; k <= S; ++k) lo[k] = (int)((long long)nsy * k / S);
      std::vector<std::pair<int, int>> order;  // (0 = Y, 1 = X, 2 = row_reduce; slab)
      for (int k = 0; k < S; ++k) {
        order.push_back({0, k});
        if (k >= 1) { order.push_back({1, k - 1}); order.push_back({2, k - 1}); }
      }
      order.push_back({1, S - 1});
      order.push_back({2, S - 1});
      for (int i = 0; i < (int)order.size(); ++i) {
        if (order[i].first == 0) iy[order[i].second] = i;
        if (order[i].first == 1) ix[order[i].second] = i;
      }
      const int rows_per_seg = s->cps[KY] * FR;
      for (int i = 0; i < (int)order.size(); ++i) {
        const int k = order[i].second, kind = order[i].first;
        KernelNode n;
        if (kind == 2) {
          const int r1 = lo[k + 1] * rows_per_seg;
          n = make_row_reduce_node(s, lo[k] * rows_per_seg, r1 < s->Ny ? r1 : s->Ny);
          n.back = {i - ix[k]};  // X_k (which waited for Y_k: the KE partials of these rows)
          st.push_back(n);
          continue;
        }
        if (!make_flow_node(s, kind ? KX : KY, kind ? cur ^ 1 : cur, &n, lo[k], lo[k + 1] - lo[k])) {
          ss_destroy(s);
          return SS_ERR_CUDA;
        }
        if (kind == 0) {
          n.back = {i + 1};  // the node before this step: the previous step's finalize
        } else {
          n.back = {i - iy[k]};
          if (k >= 1) n.back.push_back(i - iy[k - 1]);
          if (k + 1 < S) n.back.push_back(i - iy[k + 1]);
        }
        st.push_back(n);
      }
      KernelNode y, x, x0;  // the unsplit launches: ss_profile_step times these one by one
      if (!make_flow_node(s, KY, cur, &y) || !make_flow_node(s, KX, cur ^ 1, &x) ||
          !make_flow_node(s, KX, cur, &x0)) {
        ss_destroy(s);
        return SS_ERR_CUDA;
      }
      s->prof_nodes[cur].push_back(y);
      s->prof_nodes[cur].push_back(x);
      make_reduce_nodes(s, 1, s->prof_nodes[cur]);
      ev.push_back(x0);
      join = S;
    } else {
      KernelNode y, x, x0;
      if (!make_flow_node(s, KY, cur, &y) || !make_flow_node(s, s->xkind, cur ^ 1, &x) ||
          !make_flow_node(s, s->xkind, cur, &x0)) {
        ss_destroy(s);
        return SS_ERR_CUDA;
      }
      st.push_back(y);
      st.push_back(x);  // a1, a2, E, Q on the new state
      ev.push_back(x0);
    }
    make_reduce_nodes(s, 1, st, join > 1);
    if (join > 1)  // finalize waits for the row_reduce of every slab (3 nodes per slab)
      for (int k = 1; k <= 3 * join; ++k) st.back().back.push_back(k);
    make_reduce_nodes(s, 0, ev);
    if (!(s->flags & SS_FLAG_NO_GRAPH)) {
      int rc = build_graph(s, st, &s->step_exec[cur]);
      if (rc != SS_OK) { ss_destroy(s); return rc; }
    }
  }
  // MULTI steps chained in one graph: fewer launches, no inter-graph gaps.  A step that is already
  // hundreds of nodes long (demagnetisation: ~50 nodes per V-cycle) gains nothing from chaining.
  if (!(s->flags & SS_FLAG_NO_GRAPH) && s->step_nodes[0].size() <= 64) {
    for (int cur = 0; cur < 2; ++cur) {
      std::vector<KernelNode> chain;
      for (int i = 0; i < MULTI; ++i) {
        const auto& one = s->step_nodes[(cur + i) & 1];
        chain.insert(chain.end(), one.begin(), one.end());
      }
      int rc = build_graph(s, chain, &s->multi_exec[cur]);
      if (rc != SS_OK) { ss_destroy(s); return rc; }
    }
  }
  choose_resident(s);
  *out = s;
  return SS_OK;
}

int ss_destroy(ss_solver* s) {
  if (!s) return SS_ERR_ARG;
  {
    DeviceGuard guard(s);
    for (int i = 0; i < 2; ++i) {
      if (s->step_exec[i]) cudaGraphExecDestroy(s->step_exec[i]);
      if (s->multi_exec[i]) cudaGraphExecDestroy(s->multi_exec[i]);
    }
  }
  delete s;
  return SS_OK;
}

// fields go to phi(0), their frozen halo also to phi(1) (a step writes only the interior of the
// other ping-pong buffer); velocities are staged in vel(1) (host source) or read from the caller's
// array (device source) and masked to the interior into vel(0); the halo of vel(1) is zeroed.
static int set_fields_impl(ss_solver* s, const void* fields, const void* vel, cudaMemcpyKind kind) {
  if (!s || !fields) return SS_ERR_ARG;
  GUARD(s);
  const size_t nbytes = (size_t)s->batch * s->C * s->Ny * s->Nx * s->R;
  const long long planes = (long long)s->batch * s->C;
  const int grid = s->sms * 8;
  CK(cudaMemcpyAsync(s->phi(0), fields, nbytes, kind, s->stream));
  const void* vsrc = vel;
  if (vel && kind == cudaMemcpyHostToDevice) {
    CK(cudaMemcpyAsync(s->vel(1), vel, nbytes, kind, s->stream));
    vsrc = s->vel(1);
  }
  if (vsrc) {
    if (s->dtype == SS_F64)
      copy_interior_kernel<double><<<grid, 256, 0, s->stream>>>((double*)s->vel(0), (const double*)vsrc,
                                                                s->Nx, s->Ny, planes);
    else
      copy_interior_kernel<float><<<grid, 256, 0, s->stream>>>((float*)s->vel(0), (const float*)vsrc,
                                                               s->Nx, s->Ny, planes);
    s->launches += 1;
  } else {
    CK(cudaMemsetAsync(s->vel(0), 0, nbytes, s->stream));
  }
  if (s->dtype == SS_F64)
    init_halo_kernel<double><<<grid, 256, 0, s->stream>>>((double*)s->phi(1), (double*)s->vel(1),
                                                          (const double*)s->phi(0), s->Nx, s->Ny, planes);
  else
    init_halo_kernel<float><<<grid, 256, 0, s->stream>>>((float*)s->phi(1), (float*)s->vel(1),
                                                         (const float*)s->phi(0), s->Nx, s->Ny, planes);
  if (s->L.mg_bytes) CK(cudaMemsetAsync(s->ws + s->L.off_mg, 0, s->L.mg_bytes, s->stream));
  // KE partials are only written by a step: 0 after ss_set_fields
  for (int i = 0; i < 3; ++i) CK(cudaMemsetAsync(s->part(i), 0, s->L.part_bytes, s->stream));
  init_state_kernel<<<(s->batch + 127) / 128, 128, 0, s->stream>>>(s->state(), s->batch);
  s->launches += 2;
  CK(cudaGetLastError());
  s->cur = 0;
  s->steps_done = 0;
  s->fields_set = true;
  return launch_nodes(s, s->eval_nodes[0]);
}

int ss_set_fields(ss_solver* s, const void* fields_dev, const void* vel_dev) {
  return set_fields_impl(s, fields_dev, vel_dev, cudaMemcpyDeviceToDevice);
}
int ss_set_fields_host(ss_solver* s, const void* fields_host, const void* vel_host) {
  return set_fields_impl(s, fields_host, vel_host, cudaMemcpyHostToDevice);
}

// velocities are exported (zero when the last step was arrested) either into the
// caller's device array or, for a host destination, into the idle ping-pong velocity buffer,
// which the next step overwrites on the interior and never reads.
static int get_fields_impl(ss_solver* s, void* fields, void* vel, cudaMemcpyKind kind) {
  if (!s) return SS_ERR_ARG;
  if (!s->fields_set) return SS_ERR_STATE;
  GUARD(s);
  const size_t nbytes = (size_t)s->batch * s->C * s->Ny * s->Nx * s->R;
  const int grid = s->sms * 8;
  if (fields) CK(cudaMemcpyAsync(fields, s->phi(s->cur), nbytes, kind, s->stream));
  if (vel) {
    const long long per = (long long)s->C * s->Ny * s->Nx;
    void* dst = kind == cudaMemcpyDeviceToHost ? s->vel(s->cur ^ 1) : vel;
    if (s->dtype == SS_F64)
      export_velocity_kernel<double><<<grid, 256, 0, s->stream>>>(
          (double*)dst, (const double*)s->vel(s->cur), s->state(), per, s->batch);
    else
      export_velocity_kernel<float><<<grid, 256, 0, s->stream>>>(
          (float*)dst, (const float*)s->vel(s->cur), s->state(), per, s->batch);
    s->launches += 1;
    CK(cudaGetLastError());
    if (kind == cudaMemcpyDeviceToHost) CK(cudaMemcpyAsync(vel, dst, nbytes, kind, s->stream));
  }
  if (kind == cudaMemcpyDeviceToHost) CK(cudaStreamSynchronize(s->stream));
  return SS_OK;
}

int ss_get_fields(ss_solver* s, void* fields_dev, void* vel_dev) {
  return get_fields_impl(s, fields_dev, vel_dev, cudaMemcpyDeviceToDevice);
}
int ss_get_fields_host(ss_solver* s, void* fields_host, void* vel_host) {
  return get_fields_impl(s, fields_host, vel_host, cudaMemcpyDeviceToHost);
}

int ss_step(ss_solver* s, int64_t k) {
  if (!s || k < 0) return SS_ERR_ARG;
  if (!s->fields_set) return SS_ERR_STATE;
  GUARD(s);
  if (s->res_cl > 0 && k > 0) return resident_step(s, k);
  for (int64_t it = 0; it < k; ++it) {
    if (s->flags & SS_FLAG_NO_GRAPH) {
      int rc = launch_nodes(s, s->step_nodes[s->cur]);
      if (rc != SS_OK) return rc;
    } else if (k - it >= MULTI && s->multi_exec[s->cur]) {  // MULTI is even: same parity afterwards
      CK(cudaGraphLaunch(s->multi_exec[s->cur], s->stream));
      s->launches += (int64_t)MULTI * (int64_t)s->step_nodes[s->cur].size();
      s->steps_done += MULTI;
      it += MULTI - 1;
      continue;
    } else {
      CK(cudaGraphLaunch(s->step_exec[s->cur], s->stream));
      s->launches += (int64_t)s->step_nodes[s->cur].size();
    }
    s->cur ^= 1;
    s->steps_done += 1;
  }
  return SS_OK;
}

static int read_scalar(ss_solver* s, double* out, int which) {
  if (!s || !out) return SS_ERR_ARG;
  if (!s->fields_set) return SS_ERR_STATE;
  GUARD(s);
  int rc = read_state(s);
  if (rc != SS_OK) return rc;
  bool bad = false;
  for (int b = 0; b < s->batch; ++b) {
    const LatticeState& st = s->host_state[b];
    out[b] = which == 0 ? st.E : which == 1 ? st.Q : st.KE;
    bad |= st.nonfinite != 0;
  }
  return bad ? SS_ERR_NONFINITE : SS_OK;
}
int ss_energy(ss_solver* s, double* E_host) { return read_scalar(s, E_host, 0); }
int ss_charge(ss_solver* s, double* Q_host) { return read_scalar(s, Q_host, 1); }
int ss_kinetic(ss_solver* s, double* KE_host) { return read_scalar(s, KE_host, 2); }

int ss_status(ss_solver* s, int64_t* steps_done, int64_t* n_arrests, int* nonfinite) {
  if (!s) return SS_ERR_ARG;
  if (!s->fields_set) return SS_ERR_STATE;
  GUARD(s);
  int rc = read_state(s);
  if (rc != SS_OK) return rc;
  if (steps_done) *steps_done = s->steps_done;
  bool bad = false;
  for (int b = 0; b < s->batch; ++b) {
    if (n_arrests) n_arrests[b] = s->host_state[b].n_arrests;
    if (nonfinite) nonfinite[b] = s->host_state[b].nonfinite;
    bad |= s->host_state[b].nonfinite != 0;
  }
  return bad ? SS_ERR_NONFINITE : SS_OK;
}

int ss_arrests(ss_solver* s, int lattice, int64_t* steps_host, int64_t cap, int64_t* count) {
  if (!s || !count || lattice < 0 || lattice >= s->batch || cap < 0 || (cap > 0 && !steps_host))
    return SS_ERR_ARG;
  if (!s->fields_set) return SS_ERR_STATE;
  GUARD(s);
  int rc = read_state(s);
  if (rc != SS_OK) return rc;
  const int64_t total = s->host_state[lattice].n_arrests;
  *count = total;
  int64_t n = total < s->log_cap ? total : s->log_cap;
  if (n > cap) n = cap;
  if (n > 0) {
    static_assert(sizeof(long long) == sizeof(int64_t), "log entry size");
    CK(cudaMemcpyAsync(steps_host, s->ws + s->L.off_log + (size_t)lattice * s->log_cap * 8, n * 8,
                       cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
  }
  return SS_OK;
}

int ss_profile_step(ss_solver* s, int reps, double* ms_host, int cap, int* n_kernels) {
  if (!s || !ms_host || !n_kernels || reps < 1) return SS_ERR_ARG;
  if (!s->fields_set) return SS_ERR_STATE;
  GUARD(s);
  const bool split = !s->prof_nodes[0].empty();  // slab schedule: time the unsplit launches
  const int n = (int)(split ? s->prof_nodes[0] : s->step_nodes[0]).size();
  *n_kernels = n;
  if (cap < n) return SS_ERR_ARG;
  std::vector<cudaEvent_t> ev(n + 1);
  for (auto& e : ev) CK(cudaEventCreate(&e));
  std::vector<double> acc(n, 0.0);
  int rc = SS_OK;
  for (int it = 0; it < reps && rc == SS_OK; ++it) {
    auto& nodes = split ? s->prof_nodes[s->cur] : s->step_nodes[s->cur];
    cudaError_t e = cudaEventRecord(ev[0], s->stream);
    for (int i = 0; i < n && e == cudaSuccess; ++i) {
      void* params[1] = {nodes[i].args.data()};
      e = cudaLaunchKernel(nodes[i].func, nodes[i].grid, nodes[i].block, params, nodes[i].smem,
                           s->stream);
      if (e == cudaSuccess) e = cudaEventRecord(ev[i + 1], s->stream);
      s->launches += 1;
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    for (int i = 0; i < n && e == cudaSuccess; ++i) {
      float ms = 0.f;
      e = cudaEventElapsedTime(&ms, ev[i], ev[i + 1]);
      acc[i] += ms;
    }
    if (!cuda_ok(e, "ss_profile_step")) rc = SS_ERR_CUDA;
    s->cur ^= 1;
    s->steps_done += 1;
  }
  for (auto& e : ev) cudaEventDestroy(e);
  for (int i = 0; i < n; ++i) ms_host[i] = acc[i] / reps;
  return rc;
}

}  // extern "C" (templates below)

template <int THEORY, typename real>
static int render_t(ss_solver* s, int obs, int lattice, void* rgba_dev, double* minmax_host) {
  const FlowArgs<real>& fa = *reinterpret_cast<const FlowArgs<real>*>(s->consts.data());
  RenderArgs<real> r;
  memset(&r, 0, sizeof(r));
  const size_t sites = (size_t)s->Nx * s->Ny;
  r.phi = (const real*)s->phi(s->cur) + (size_t)lattice * s->C * sites;
  r.nblocks = (int)((sites + 255) / 256);
  r.part = (double*)(s->ws + s->L.off_render);
  r.minmax = r.part + 2 * (size_t)r.nblocks;
  r.nonfinite = (int*)(r.minmax + 2);
  r.rgba = (unsigned int*)rgba_dev;
  r.Nx = s->Nx; r.Ny = s->Ny; r.obs = obs;
  r.B = real(s->Bb_host[lattice]);
  CK(cudaMemsetAsync(r.nonfinite, 0, sizeof(int), s->stream));
  observable_kernel<THEORY, real><<<r.nblocks, 256, 0, s->stream>>>(fa, r);
  minmax_kernel<real><<<1, 1024, 0, s->stream>>>(r);
  colormap_kernel<THEORY, real><<<r.nblocks, 256, 0, s->stream>>>(fa, r);
  s->launches += 3;
  CK(cudaGetLastError());
  if (minmax_host) {
    double out[3];  // min, max, flag word
    CK(cudaMemcpyAsync(out, r.minmax, 3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    minmax_host[0] = out[0];
    minmax_host[1] = out[1];
    int flag;
    memcpy(&flag, &out[2], sizeof(int));
    if (flag) return SS_ERR_NONFINITE;
  }
  return SS_OK;
}

extern "C" {

int ss_render(ss_solver* s, int observable, int lattice, void* rgba_dev, double* minmax_host) {
  if (!s || !rgba_dev || lattice < 0 || lattice >= s->batch || observable < 0 || observable > 2)
    return SS_ERR_ARG;
  if (!s->fields_set) return SS_ERR_STATE;
  GUARD(s);
  const bool f64 = s->dtype == SS_F64;
  switch (s->ktheory) {
    case kCM: return f64 ? render_t<kCM, double>(s, observable, lattice, rgba_dev, minmax_host)
                         : render_t<kCM, float>(s, observable, lattice, rgba_dev, minmax_host);
    case kAH: return f64 ? render_t<kAH, double>(s, observable, lattice, rgba_dev, minmax_host)
                         : render_t<kAH, float>(s, observable, lattice, rgba_dev, minmax_host);
    case kBS: return f64 ? render_t<kBS, double>(s, observable, lattice, rgba_dev, minmax_host)
                         : render_t<kBS, float>(s, observable, lattice, rgba_dev, minmax_host);
    default:  return f64 ? render_t<kCMG, double>(s, observable, lattice, rgba_dev, minmax_host)
                         : render_t<kCMG, float>(s, observable, lattice, rgba_dev, minmax_host);
  }
}

const char* ss_schedule_name(const ss_solver* s) {
  if (!s) return "";
  if (s->res_cl > 0) return "resident-cluster";
  if (s->ktheory == kBS) return "per-stage tile kernels";
  if (s->demag != 0.0) return "pointwise kernels + multigrid V-cycles";
  if (s->slabs > 1) return "two-kernel, row slabs";
  return s->integrator == SS_VERLET ? "one-kernel verlet" : "two-kernel";
}

const char* ss_kernel_name(const ss_solver* s, int i) {
  if (!s) return "";
  const auto& nodes = s->prof_nodes[0].empty() ? s->step_nodes[0] : s->prof_nodes[0];
  return i >= 0 && i < (int)nodes.size() ? nodes[i].name : "";
}

int64_t ss_launch_count(const ss_solver* s) { return s ? s->launches : 0; }

const char* ss_strerror(int code) {
  switch (code) {
    case SS_OK: return "ok";
    case SS_ERR_ARG: return "invalid argument";
    case SS_ERR_UNSUPPORTED: return "unsupported request";
    case SS_ERR_CUDA: return g_cuda_msg[0] ? g_cuda_msg : "CUDA failure";
    case SS_ERR_WORKSPACE: return "workspace missing, too small or misaligned";
    case SS_ERR_STATE: return "fields not set";
    case SS_ERR_NONFINITE: return "non-finite energy";
    case SS_ERR_TOO_LARGE: return "lattice exceeds SS_NOALLOC_MAX_SITES (2048 x 2048 sites) of ss_render_noalloc";
    default: return "unknown status";
  }
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Allocation-free entry point (include/ss.h ss_render_noalloc): the render kernels of
// ss_render.cuh with their scratch -- the per-block extrema and the non-finite flag -- in a
// file-scope device array instead of a caller workspace, so that no handle (ss_create builds
// CUDA graphs, i.e. allocates) and no workspace is needed.  Every call on a device shares the
// array; calls that overlap on the GPU race on it.
namespace {

constexpr long long NOALLOC_MAX_SITES = SS_NOALLOC_MAX_SITES;
constexpr int NOALLOC_MAX_BLOCKS = (int)((NOALLOC_MAX_SITES + 255) / 256);
constexpr int NOALLOC_FLAG_AT = 2 * NOALLOC_MAX_BLOCKS;  // the flag word sits after the partials
constexpr int NOALLOC_MAX_DEVICES = 64;
// [2 * NOALLOC_MAX_BLOCKS] block (min, max), then the non-finite flag: 256 KiB + 256 B per device
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_FLAG_AT + 32];

// In host code `g_noalloc_scratch` is only a stand-in for the symbol; the device address is
// looked up once per device, with that device current, and cached here.
double* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};
std::mutex g_noalloc_mutex;

int noalloc_scratch(int device, double** out) {
  if (device < 0 || device >= NOALLOC_MAX_DEVICES) return SS_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[device]) {
    double* ptr = nullptr;  // the caller has made `device` current
    if (!cuda_ok(cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch), "cudaGetSymbolAddress") ||
        !ptr)
      return SS_ERR_CUDA;
    g_noalloc_ptr[device] = ptr;
  }
  *out = g_noalloc_ptr[device];
  return SS_OK;
}

template <int THEORY, typename real>
int render_noalloc_t(const ss_solver* k, double* scratch, int obs, const void* fields_dev,
                     void* rgba_dev, double* minmax_dev, int* nonfinite_dev) {
  FlowArgs<real> fa;
  memset(&fa, 0, sizeof(fa));
  fill_constants(k, fa);
  RenderArgs<real> r;
  memset(&r, 0, sizeof(r));
  const size_t sites = (size_t)k->Nx * k->Ny;
  r.phi = (const real*)fields_dev;
  r.nblocks = (int)((sites + 255) / 256);
  r.part = scratch;
  r.minmax = minmax_dev;
  r.nonfinite = (int*)(scratch + NOALLOC_FLAG_AT);
  r.rgba = (unsigned int*)rgba_dev;
  r.Nx = k->Nx; r.Ny = k->Ny; r.obs = obs;
  r.B = real(k->B);
  // the array keeps the last call's contents: the flag must start at zero (the block partials
  // [0, 2 nblocks) are all rewritten by observable_kernel before minmax_kernel reads them)
  CK(cudaMemsetAsync(r.nonfinite, 0, sizeof(int), k->stream));
  observable_kernel<THEORY, real><<<r.nblocks, 256, 0, k->stream>>>(fa, r);
  minmax_kernel<real><<<1, 1024, 0, k->stream>>>(r);
  if (rgba_dev) colormap_kernel<THEORY, real><<<r.nblocks, 256, 0, k->stream>>>(fa, r);
  CK(cudaGetLastError());
  if (nonfinite_dev)
    CK(cudaMemcpyAsync(nonfinite_dev, r.nonfinite, sizeof(int), cudaMemcpyDeviceToDevice, k->stream));
  return SS_OK;
}

}  // namespace

extern "C" int ss_render_noalloc(int theory, int Nx, int Ny, double h, const ss_params* p,
                                 int observable, const void* fields_dev, void* rgba_dev,
                                 double* minmax_dev, int* nonfinite_dev) {
  if (!p || !fields_dev || !minmax_dev || observable < 0 || observable > 2) return SS_ERR_ARG;
  ss_params q = *p;
  q.batch = 1;  // one lattice per call; workspace, B_batch, integrator and flags are not used
  q.flags = 0;
  if (!valid_shape(theory, Nx, Ny, &q) || !(h > 0.0) || !std::isfinite(h)) return SS_ERR_ARG;
  if (theory == SS_THEORY_BABY_SKYRME && p->dmi_d) return SS_ERR_UNSUPPORTED;
  if ((long long)Nx * Ny > NOALLOC_MAX_SITES) return SS_ERR_TOO_LARGE;
  cudaPointerAttributes pa;
  if (!cuda_ok(cudaPointerGetAttributes(&pa, fields_dev), "cudaPointerGetAttributes"))
    return SS_ERR_CUDA;
  if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return SS_ERR_ARG;
  ss_solver k;  // host-side carrier of the constants only (never stepped, owns nothing)
  k.theory = theory; k.dtype = p->dtype; k.Nx = Nx; k.Ny = Ny; k.batch = 1; k.h = h;
  k.device = pa.device;
  k.dt = 0.5 * h;
  k.kappa = p->kappa; k.B = p->B; k.K = p->K; k.lambda = p->lambda;
  k.mu = p->mu; k.pot = p->potential; k.potN = p->potential_n;
  k.stream = (cudaStream_t)p->stream;
  k.L.nseg = (Nx + SEG - 1) / SEG;
  k.ktheory = theory == SS_THEORY_BABY_SKYRME ? kBS : theory;
  for (int i = 0; i < 6; ++i) k.dmi[i] = 0.0;
  if (theory == SS_THEORY_CHIRAL_MAGNET && p->dmi_d) {
    k.ktheory = kCMG;
    for (int i = 0; i < 6; ++i) {
      if (!std::isfinite(p->dmi_d[i])) return SS_ERR_ARG;
      k.dmi[i] = p->dmi_d[i];
    }
  }
  GUARD(&k);
  double* scratch = nullptr;
  int rc = noalloc_scratch(k.device, &scratch);
  if (rc != SS_OK) return rc;
  const bool f64 = p->dtype == SS_F64;
#define SS_NOALLOC_CASE(TH)                                                                        \
  return f64 ? render_noalloc_t<TH, double>(&k, scratch, observable, fields_dev, rgba_dev,         \
                                            minmax_dev, nonfinite_dev)                             \
             : render_noalloc_t<TH, float>(&k, scratch, observable, fields_dev, rgba_dev,          \
                                           minmax_dev, nonfinite_dev)
  switch (k.ktheory) {
    case kCM: SS_NOALLOC_CASE(kCM);
    case kAH: SS_NOALLOC_CASE(kAH);
    case kBS: SS_NOALLOC_CASE(kBS);
    default:  SS_NOALLOC_CASE(kCMG);
  }
#undef SS_NOALLOC_CASE
}
