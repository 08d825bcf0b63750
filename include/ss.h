/*
 * ss.h — C ABI of libss.so: the arrested-Newton-flow energy-minimisation step of
 * arxiv/paper_2603_24370 (soliton_solver) on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (citations: /root/reference/PAPER.md line numbers; "DESIGN Rn"
 * = reading n in DESIGN.md where the paper is silent):
 *   - a rectangular 2-D lattice with a frozen halo of width two and the 4th-order central
 *     stencils of PAPER.md:100-109 (eq. 1, eq. 2);
 *   - the discretised energy E_h, its exact gradient and the topological charge of
 *       SS_THEORY_CHIRAL_MAGNET  n in S^2:  1/2|grad n|^2 + kappa n.(curl n) + B(1-n3) + K(1-n3^2)
 *                                (PAPER.md:196 eq. 5, :327; DESIGN R1-R3); optionally the DMI
 *                                term as kappa sum_mu d_mu.(n x d_mu n) with a table (dmi_d,
 *                                DESIGN R16) and the magnetostatic energy (g/2)|grad psi|^2,
 *                                lap psi = div n (demag; eq. 5-6; DESIGN R19),
 *       SS_THEORY_ABELIAN_HIGGS  phi in C, A in R^2: 1/2|D phi|^2 + 1/2 (curl A)^2
 *                                + (lambda/8)(1-|phi|^2)^2   (DESIGN R1-R3, R9),
 *       SS_THEORY_BABY_SKYRME    m in S^2: 1/2|grad m|^2 + (kappa^2/2)|d1 m x d2 m|^2 + V(m)
 *                                (DESIGN R18; C = 3, charge = degree as for
 *                                the chiral magnet);
 *   - the arrested Newton flow phi'' = -grad E_h (eq. 3) integrated with
 *     classical RK4, the unit-length projection applied in every stage
 *     (PAPER.md:129+154), the velocity set to zero whenever E_h rises (eq. 4);
 *   - device-resident reductions of E, Q and the kinetic energy in a fixed tree order
 *     (DESIGN R10) that drive the arrest with no host synchronisation.
 *
 * Conventions
 *   Lattice   Nx x Ny sites INCLUDING the halo (DESIGN R4); site (i,j), i fastest.
 *             Interior = 2 <= i < Nx-2, 2 <= j < Ny-2.  Halo sites are frozen: supplied by
 *             ss_set_fields and never written by a step.
 *   Layout    field arrays are dense [batch][C][Ny][Nx] of `real` (double for SS_F64, float
 *             for SS_F32), x fastest.  C = 3 (n1,n2,n3) for the chiral magnet and baby Skyrme, C = 4
 *             (Re phi, Im phi, A1, A2) for Abelian Higgs.  Velocities have the same shape;
 *             their halo entries are ignored on input and written as 0 on output.
 *   Memory    every pointer named *_dev is DEVICE memory owned by the caller; every pointer
 *             named *_host is HOST memory owned by the caller.  The library allocates no
 *             device memory: all of its state lives in the caller's `workspace`
 *             (ss_workspace_bytes), which must outlive the handle (the only device memory of
 *             its own is the static 256 KiB scratch array of ss_render_noalloc).  The caller
 *             also owns the CUDA stream; all work is enqueued on it.
 *   Errors    every call returns an SS_* status; nothing throws or aborts across the ABI.
 *   Threads   a handle is not thread-safe; distinct handles are independent.
 *   No CPU fallback exists: without a CUDA device ss_create returns SS_ERR_CUDA.
 */
#ifndef SS_H_
#define SS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ss_solver ss_solver; /* opaque */

enum { SS_THEORY_CHIRAL_MAGNET = 0, SS_THEORY_ABELIAN_HIGGS = 1, SS_THEORY_BABY_SKYRME = 2 };
/* baby-Skyrme potentials (PAPER.md:90 names them, no formula is printed; DESIGN R18), vacuum e3:
 *   SS_POT_STANDARD    V = mu^2 (1 - m3)
 *   SS_POT_EASY_PLANE  V = 1/2 mu^2 m1^2
 *   SS_POT_BROKEN      V = mu^2 |1 - (m1 + i m2)^N|^2 (1 - m3),  N = potential_n in 1..16 */
enum { SS_POT_STANDARD = 0, SS_POT_EASY_PLANE = 1, SS_POT_BROKEN = 2 };
enum { SS_F64 = 0, SS_F32 = 1 };
enum {
  SS_OK = 0,
  SS_ERR_ARG = -1,         /* NULL pointer, bad size/enum, misaligned row length           */
  SS_ERR_UNSUPPORTED = -2, /* valid request this build does not implement                   */
  SS_ERR_CUDA = -3,        /* CUDA runtime failure (text via ss_strerror)                   */
  SS_ERR_WORKSPACE = -4,   /* workspace NULL / too small / misaligned                       */
  SS_ERR_STATE = -5,       /* stepping or reading before ss_set_fields                      */
  SS_ERR_NONFINITE = -6,   /* an energy became NaN/Inf (values are still written)           */
  SS_ERR_TOO_LARGE = -7    /* ss_render_noalloc: Nx * Ny exceeds SS_NOALLOC_MAX_SITES       */
};

/* Integrators.  SS_RK4 is the paper's example ("such as fourth-order Runge-Kutta").
 * SS_VERLET is the one-gradient-per-step variant (DESIGN R15): velocity Verlet
 *   w = vh + dt/2 a(phi), phi' = R(phi + dt w), v' = Pi(w + dt/2 a(phi'))
 * with the same projection (PAPER.md:129+154) and the same arrest (eq. 4). */
enum { SS_RK4 = 0, SS_VERLET = 1 };

/* ss_params.flags (debugging aid, not part of the method) */
enum { SS_FLAG_NO_GRAPH = 1,   /* launch the step's kernels one by one instead of replaying the
                                  per-step CUDA graphs; results are bitwise identical */
       SS_FLAG_NO_RESIDENT = 2,/* never use the resident-cluster schedule (see ss_step); results
                                  are bitwise identical */
       SS_FLAG_NO_SLABS = 4    /* never split the RK4 step's two kernels into row slabs that
                                  overlap inside the graph (see ss_step); results are bitwise
                                  identical */ };

typedef struct {
  int dtype;               /* SS_F64 | SS_F32: field storage and per-site arithmetic;       */
                           /* reductions, E, Q, KE and the arrest test are always fp64      */
  int batch;               /* 1..65535 independent lattices sharing Nx, Ny, h, dt           */
  double dt;               /* <= 0 -> 0.5*h (Courant number C = 0.5)          */
  double kappa, B, K;      /* chiral magnet: DMI, Zeeman field, uniaxial anisotropy         */
  const double* B_batch;   /* optional HOST array[batch]: per-lattice B (overrides B)       */
  double lambda;           /* Abelian Higgs coupling (critical at 1)                        */
  void* workspace;         /* DEVICE memory, >= ss_workspace_bytes, 256-byte aligned; the   */
                           /* solver runs on the device this memory lives on                */
  size_t workspace_bytes;
  void* stream;            /* cudaStream_t of that device, owned by the caller; NULL =      */
                           /* default stream                                                */
  int64_t arrest_log_capacity; /* entries per lattice; 0 -> 4096; later arrests are counted */
                               /* but not logged                                            */
  int integrator;          /* SS_RK4 | SS_VERLET                                            */
  int flags;               /* 0 or a combination of SS_FLAG_*                                */
  int chunks_per_segment;  /* tuning, 0 = auto: rows/4 each CTA of the flow kernels marches */
                           /* (results do not depend on it)                                 */
  const double* dmi_d;     /* chiral magnet, optional HOST array[6] = (d_x, d_y): the DMI term   */
                           /* kappa sum_mu d_mu.(n x d_mu n) of PAPER.md:196 eq. (5) (DESIGN    */
                           /* R16).  NULL = kappa n.(curl n), i.e. d_x = -e_x, d_y = -e_y       */
  double mu;               /* baby Skyrme: V is proportional to mu^2 (kappa = Skyrme coupling)   */
  int potential;           /* baby Skyrme: SS_POT_*                                              */
  int potential_n;         /* baby Skyrme: N of SS_POT_BROKEN                                    */
  double demag;            /* chiral magnet: g = mu0 Ms^2 >= 0 of the magnetostatic energy           */
                           /* (g/2)|grad psi|^2, lap psi = d1 n1 + d2 n2, psi = 0 on the halo         */
                           /* (PAPER.md:196 eq. 5, :199-203 eq. 6; DESIGN R19); 0 = off.  Needs       */
                           /* SS_F64; psi is solved by multigrid V-cycles on the device: one solve    */
                           /* per step with SS_VERLET, one per RK4 stage field (four) with SS_RK4     */
  int demag_cycles;        /* V-cycles per solve, warm-started (0 -> 8; 4x as many in ss_set_fields);  */
                           /* measured contraction per cycle 0.27                                     */
} ss_params;

/* Limits of this build: 5 <= Nx <= 65536, 5 <= Ny <= 32768 (the device-side reduction tree of
 * PAPER.md:158 / DESIGN R10 is finished by one warp per row and one CTA per lattice),
 * 1 <= batch <= 65535; Nx even for SS_F64 and a multiple of 4 for SS_F32 (16-byte rows).
 * Breaking an alignment or lower bound is SS_ERR_ARG, exceeding an upper bound is
 * SS_ERR_UNSUPPORTED. */

/* Bytes of device workspace ss_create needs for this problem (fields, velocities,
 * accelerations of the Runge-Kutta stages, reduction buffers -- here two copies of phi and v, two
 * acceleration arrays, partial sums, per-lattice state, arrest logs).  Returns 0 when ss_create
 * would refuse the arguments (invalid or over a limit); p->workspace may be NULL here. */
size_t ss_workspace_bytes(int theory, int Nx, int Ny, const ss_params* p);

/* Create a solver (lattice, spacing, components and time step are fixed
 * before any device buffer is carved).  *out is NULL on failure.  The solver is bound to the
 * device of p->workspace; every later call may be made with any device current. */
int ss_create(ss_solver** out, int theory, int Nx, int Ny, double h, const ss_params* p);
/* Release the handle (the device buffers are the caller's workspace and stream,
 * which this call leaves untouched).  Pending work on the stream is not waited for. */
int ss_destroy(ss_solver* s);

/* Load fields (halo included, frozen from now on) and velocities (NULL = from rest,
 * PAPER.md:123) by device-to-device copies on the stream; resets the step counter and the
 * arrest log, sets E_prev = +inf (step 0 cannot arrest) and evaluates a(phi), E, Q so that
 * ss_energy / ss_charge are valid at once.  |n| = 1 is NOT enforced on input. */
int ss_set_fields(ss_solver* s, const void* fields_dev, const void* vel_dev);

/* Copy the current fields / velocities out (either may be NULL).  After an arrested step
 * the velocity reads as exactly 0. */
int ss_get_fields(ss_solver* s, void* fields_dev, void* vel_dev);

/* The same two calls for HOST arrays (same layout and semantics; pinned memory makes the
 * copies asynchronous).  The transfers go straight to / from the workspace on the stream;
 * ss_get_fields_host synchronises the stream before returning. */
int ss_set_fields_host(ss_solver* s, const void* fields_host, const void* vel_host);
int ss_get_fields_host(ss_solver* s, void* fields_host, void* vel_host);

/* Enqueue k flow steps (asynchronous; no host synchronisation, the arrest of eq. 4 is
 * decided on the device; the steps are CUDA-graph replays, 8 steps per graph launch plus
 * single-step graphs for the remainder; steps of more than 64 kernels -- demagnetisation -- are
 * replayed one step per graph launch).  One step = RK4 stages 2-4 + update + projection, then the
 * stencil pass on the new field (a, E, Q) and the arrest decision.
 * Small lattices (fp64 chiral magnet, SS_RK4, Nx a multiple of 32, the whole state within the
 * shared memory of one thread-block cluster per lattice, e.g. 64 x 64 ... 128 x 128) take all k
 * steps in ONE launch with the state resident in shared memory; fields, E, Q, KE and the arrest
 * log are bitwise identical to the general schedule.
 * Large lattices (SS_RK4, at least two waves of CTAs and eight row segments per lattice: from
 * about 1536 x 1536 sites, or a few batched 512 x 512 ones) have the step's two flow kernels
 * split into four row slabs each, joined in the graph by the data dependencies only, so that
 * the second kernel starts on the rows the first has finished; again bitwise identical
 * (SS_FLAG_NO_SLABS). */
int ss_step(ss_solver* s, int64_t k);

/* Scalar read-outs: synchronise the stream, then fill HOST arrays of length batch.
 * Return SS_ERR_NONFINITE (after filling) if any lattice has a non-finite energy.
 *   ss_energy   E_h[phi] of the current field: h^2 times the canonical-tree sum of the site-form
 *               energy densities (PAPER.md:117 "discretized energy functional", :158 "total
 *               energy ... parallel GPU reductions"; DESIGN R1, R3, R10).
 *   ss_charge   topological charge ("conserved topological charge"; DESIGN R9):
 *               CM degree (1/4 pi) h^2 sum n.(D_x n x D_y n), AH flux / 2 pi, same tree.
 *   ss_kinetic  1/2 h^2 sum |v|^2 of the last step before its arrest ("kinetic
 *               energy"; diagnostic, DESIGN R10); 0 after ss_set_fields. */
int ss_energy(ss_solver* s, double* E_host);
int ss_charge(ss_solver* s, double* Q_host);
int ss_kinetic(ss_solver* s, double* KE_host);
/* State of the arrest logic of PAPER.md:125-127 eq. (4).  steps_done: scalar; n_arrests,
 * nonfinite: HOST arrays[batch]; any may be NULL.  Synchronises the stream. */
int ss_status(ss_solver* s, int64_t* steps_done, int64_t* n_arrests, int* nonfinite);
/* Arrest log of one lattice (eq. 4; DESIGN R8): the 1-based indices n+1 of
 * the steps whose result raised the energy.  Writes min(count, cap, arrest_log_capacity)
 * entries to steps_host (HOST), the total number of arrests to *count. */
int ss_arrests(ss_solver* s, int lattice, int64_t* steps_host, int64_t cap, int64_t* count);

/* Headless visualisation (DESIGN R17): writes the image
 * of one observable of lattice `lattice` as [Ny][Nx] RGBA8 words (R in the low byte) into
 * rgba_dev (DEVICE memory), mapped linearly between the observable's extrema over the finite
 * interior values, which a device-side reduction finds; halo sites are 0 (transparent), a
 * non-finite interior value is opaque magenta.  minmax_host (HOST array[2], may be NULL)
 * receives the extrema and makes the call synchronise the stream; only then can the call
 * report SS_ERR_NONFINITE (image and extrema are still written).  No window, no GL interop. */
enum { SS_OBS_ENERGY = 0,   /* site-form energy density e_i                                   */
       SS_OBS_CHARGE = 1,   /* CM: degree density; AH: flux density / 2 pi                     */
       SS_OBS_ORDER = 2 };  /* CM: n3; AH: |phi| (order-parameter magnitude)                   */
int ss_render(ss_solver* s, int observable, int lattice, void* rgba_dev, double* minmax_host);

/* Allocation-free variant of ss_render (the same operation: device-side
 * extrema and the colour-mapped image of an observable; DESIGN R17) for callers that cannot
 * allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): no handle
 * -- ss_create instantiates CUDA graphs -- and no workspace.  The same kernels as ss_render on
 * ONE lattice fields_dev (DEVICE, [C][Ny][Nx], dtype p->dtype), with their scratch (per-block
 * extrema, non-finite flag) in a static device array inside the library: 256 KiB + 256 B that
 * every GPU which loads the library holds until exit, sized for Nx * Ny <= SS_NOALLOC_MAX_SITES
 * (larger lattices: SS_ERR_TOO_LARGE).  Read from p: dtype, kappa, B,
 * K, lambda, dmi_d, mu, potential, potential_n, stream; everything else is ignored.  Outputs,
 * all DEVICE memory of the caller: rgba_dev [Ny][Nx] RGBA8 (may be NULL: extrema only),
 * minmax_dev double[2], nonfinite_dev int[1] (may be NULL; 1 when an interior value was NaN or
 * Inf).  Asynchronous on p->stream: one 4-byte memset, two or three kernels, one 4-byte
 * device-to-device copy; calls cudaMalloc, cudaFree or an allocating library routine never.
 * The first call on a device looks up the array's address (cudaGetSymbolAddress, which may load
 * the module): make one call per device before capturing.  All calls on a device share the
 * array, which keeps the last call's contents (the call clears what must start at zero): calls
 * that overlap on the GPU -- different streams, or graphs replayed concurrently -- race. */
#define SS_NOALLOC_MAX_SITES (2048 * 2048)
int ss_render_noalloc(int theory, int Nx, int Ny, double h, const ss_params* p, int observable,
                      const void* fields_dev, void* rgba_dev, double* minmax_dev,
                      int* nonfinite_dev);

const char* ss_strerror(int code);

/* ---------------------------------------------------------------------------------------------
 * Measurement-only entry points (used by bench.py and the tests; not part of the method).
 * --------------------------------------------------------------------------------------------- */

/* Number of kernel launches (graph nodes included) enqueued by this handle so far. */
int64_t ss_launch_count(const ss_solver* s);

/* Run `reps` real flow steps launching the step's kernels one by one with a CUDA event between
 * consecutive launches on the solver's stream, and return the average device time of each
 * kernel in milliseconds (HOST array, `cap` entries; *n_kernels = number of kernels in one
 * step, in launch order; ss_kernel_name(i) names entry i).  The state advances by `reps` steps
 * exactly as with ss_step(reps).  Synchronises the stream. */
int ss_profile_step(ss_solver* s, int reps, double* ms_host, int cap, int* n_kernels);
const char* ss_kernel_name(const ss_solver* s, int i);
/* Name of the schedule ss_step uses for this solver ("two-kernel", "resident-cluster", ...). */
const char* ss_schedule_name(const ss_solver* s);

#ifdef __cplusplus
}
#endif
#endif /* SS_H_ */
