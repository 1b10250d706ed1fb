/* ep.h -- C-ABI of libep: the explicit monodomain + ten Tusscher-Panfilov 2006 time step of
 * arXiv 2112.12854 (section 3.2) on a tetrahedral cell-centred finite-volume mesh, one B200 (sm_100a), fp64.
 *
 * Citations are PAPER.md:<line> (section / equation).  Readings of silent or ambiguous points (A1..A18, B1..B9) are
 * listed in DESIGN.md section 3.
 *
 * Conventions
 *   - every function returns EP_OK (0) or a negative error code and never throws across the ABI;
 *     ep_last_error() returns a thread-local, NUL-terminated message for the last failing call of this thread;
 *   - all pointer arguments are HOST pointers unless the comment says "device"; inputs are copied before the call
 *     returns (the caller may free them), outputs are written into caller-owned buffers;
 *   - cells and nodes keep the CALLER's numbering at the ABI: the space-filling-curve permutation used on the device
 *     is invisible except through ep_device_vm();
 *   - one handle is used by one thread at a time; there is no global state besides the error string;
 *   - there is no CPU fallback: without a CUDA device ep_mesh_create() fails with EP_ERR_CUDA.
 *     (ep_host_stencil() runs the one-time host preprocessor only and needs no device; it exists so that the
 *     host logic can be tested on a machine without a GPU.)
 *   - units: lengths mm, conductivities mS/cm, chi 1/cm, Cm uF/cm^2, potentials mV, time ms, stimulus uA/cm^2
 *     (PAPER.md:113 gives the same physics in mm units: chi = 140 1/mm, Cm = 0.01 uF/mm^2; reading A14).
 */
#ifndef EP_H_
#define EP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ep_sim ep_sim; /* opaque; owns all host and device memory it allocates */

enum { EP_OK = 0, EP_ERR_ARG = -1, EP_ERR_MESH = -2, EP_ERR_STATE = -3, EP_ERR_CUDA = -4, EP_ERR_NOMEM = -5,
       EP_ERR_NUMERIC = -6 };
enum { EP_MODEL_TP06 = 0, EP_MODEL_CRN98 = 1, EP_MODEL_STEWART = 2 };
enum { EP_MAX_STIM_SLOTS = 8 };

/* Number of state variables of a cell model, Vm included (TP06 19, Courtemanche 21, Stewart 20); <0 if
 * unknown. */
int ep_model_n_states(int model);

/* Build the simulation object: validate the mesh, run the one-time preprocessor (geometry, face matching, node stars,
 * the Fig. 8 a->e pipeline of PAPER.md:164-168 with the eq. (8) correction folded into per-cell gather coefficients,
 * Morton reordering, ELL packing) and upload the tables.
 *   xyz_mm       [n_nodes*3] node coordinates, mm
 *   tets         [n_tets*4]  0-based node ids, any orientation
 *   fibre        [n_tets*3]  per-cell fibre direction (normalised inside); NULL => isotropic sigma_l
 *   sigma_scale  [n_tets]    per-cell multiplier of the conductivity tensor (PAPER.md:309 pathologies); NULL => 1
 *   sigma_l/t    mS/cm, M_c = scale*[sigma_t I + (sigma_l - sigma_t) f f^T]  (eq. (2)-(3))
 *   chi, Cm      surface-to-volume ratio 1/cm and membrane capacitance uF/cm^2
 * Errors: EP_ERR_ARG (NULL/negative sizes, non-positive sigma/chi/Cm), EP_ERR_MESH (index out of range, zero volume,
 * face shared by >2 cells, non-finite coordinate, zero fibre vector), EP_ERR_CUDA, EP_ERR_NOMEM.  *out is NULL on error. */
int ep_mesh_create(ep_sim **out, int64_t n_nodes, const double *xyz_mm, int64_t n_tets, const int32_t *tets,
                   const double *fibre, const double *sigma_scale, double sigma_l, double sigma_t, double chi,
                   double Cm);

/* The same for a two-dimensional medium (the Purkinje network): a triangulated surface embedded in 3D,
 * tris [n_tris*3].  PAPER.md:170: "a similar FV approach is used to discretize the ... equations over 1D and 2D media": the
 * chain of PAPER.md:164-168 with edges for faces, edge lengths for face areas and triangle areas for cell volumes (a uniform
 * layer thickness cancels); readings D1-D3 of DESIGN.md section 3.  Every other call works on the handle unchanged ("n_tets"
 * then means the number of triangles, ep_mean_vm is area-weighted).  Errors as ep_mesh_create; EP_ERR_MESH also for an edge
 * shared by more than two triangles. */
int ep_mesh_create_tri(ep_sim **out, int64_t n_nodes, const double *xyz_mm, int64_t n_tris, const int32_t *tris,
                       const double *fibre, const double *sigma_scale, double sigma_l, double sigma_t, double chi,
                       double Cm);

/* Bidomain model, eq. (1) / (6) of the paper: intracellular and extracellular conductivities along /
 * across the fibres in mS/cm (Table 2: 1.7 / 0.19 and 6.2 / 2.4).  Time stepping as PAPER.md:176-178: ep_step
 * advances v explicitly from v, v_ext, I_ion, I_s at t^n with the fused kernel (the term div(M_int grad v_ext) enters as a
 * per-cell source), then solves  div((M_int + M_ext) grad v_ext) = -div(M_int grad v)  for v_ext at t^{n+1} by restarted GMRES
 * entirely on the device, first estimate = v_ext of the previous step.  Readings E1-E4 of DESIGN.md: the system is singular
 * under no-flux boundaries and v_ext is the solution with zero volume-weighted mean; v_ext at t = 0 solves the same equation
 * for the initial potential; defaults restart 30, relative residual 1e-10, no preconditioner.  Tetrahedra only.
 * A solve that does not reach the tolerance within max_cycles restarts sets the sticky error EP_ERR_NUMERIC. */
int ep_mesh_create_bidomain(ep_sim **out, int64_t n_nodes, const double *xyz_mm, int64_t n_tets, const int32_t *tets,
                            const double *fibre, const double *sigma_scale, double sigma_int_l, double sigma_int_t,
                            double sigma_ext_l, double sigma_ext_t, double chi, double Cm);
/* Solver settings: restart length in [1, 63], restarts allowed per solve, relative residual |b - A x| / |b|. */
int ep_bidomain_solver(ep_sim *sim, int restart, int max_cycles, double rel_tol);
/* Extracellular potential at the current time, [n_tets] in the caller's order, zero volume-weighted mean; synchronises. */
int ep_read_vext(ep_sim *sim, double *out);
/* GMRES iterations of the last solve / of all solves, number of solves, last relative residual; any pointer may be NULL. */
int ep_bidomain_stats(ep_sim *sim, int64_t *iters_last, int64_t *iters_total, int64_t *solves, double *rel_res_last);

/* Intra-mesh sharding (the paper itself uses one GPU per chamber).  The cells of ONE mesh are
 * cut into n_parts contiguous ranges of the Morton curve through their centroids.  Part p owns one range and keeps, as halo,
 * every other cell within two node-rings of an owned cell -- the reach of the stencil (the nodes of a cell and
 * of its face neighbours, and the cells around those nodes).  ep_step advances the owned cells only; between two steps every
 * part needs the new Vm of its halo cells from their owners: one neighbour exchange per step, no global reduction.
 *
 * ep_shard_create takes the GLOBAL mesh (every rank holds it on the host) and builds part `part`: a handle whose cells are
 * numbered locally -- owned cells first (ascending global id), then halo cells (ascending global id); every other call
 * (ep_state_init, ep_stimulus_set, ep_read_vm ...) works in that local numbering with n_tets = n_local.  Values read back for
 * halo cells are the last received copies; activation times and ep_mean_vm cover the owned cells (ep_mean_vm: owned volume
 * weights, so the global mean is the volume-weighted mean of the parts').
 * ep_shard_info: sizes, the global id of every local cell [n_local], and the per-peer segments [n_parts+1] of the two
 * exchange buffers (any pointer may be NULL).  The segment a part sends to peer q lists the same cells in the same order
 * (ascending global id) as q's receive segment from that part.
 * ep_shard_buffers: DEVICE pointers of the send / receive buffers (doubles), for NCCL send/recv or peer copies.
 * One step of a sharded run: ep_step(sim, 1, dt); ep_halo_pack(sim); <exchange the segments>; ep_halo_unpack(sim).
 * ep_halo_exchange_local does pack + exchange + unpack for all parts living in ONE process (device-to-device copies).
 * ep_shard_plan is the host-only partitioner (no device needed): counts[4] = {n_owned, n_local, n_send, n_recv}, local_cells
 * [n_local], send/recv segment pointers [n_parts+1] and the cells of both buffers as GLOBAL ids; arrays of capacity n_tets are
 * always large enough; any of them may be NULL.  n_parts <= 64.  Not available for bidomain handles. */
int ep_shard_plan(int64_t n_nodes, const double *xyz_mm, int64_t n_tets, const int32_t *tets, int part, int n_parts,
                  int64_t *counts, int64_t *local_cells, int64_t *send_ptr, int64_t *send_global, int64_t *recv_ptr,
                  int64_t *recv_global);
int ep_shard_create(ep_sim **out, int64_t n_nodes, const double *xyz_mm, int64_t n_tets, const int32_t *tets,
                    const double *fibre, const double *sigma_scale, double sigma_l, double sigma_t, double chi, double Cm,
                    int part, int n_parts);
int ep_shard_info(ep_sim *sim, int64_t *n_owned, int64_t *n_local, int64_t *global_ids, int64_t *send_ptr, int64_t *recv_ptr);
int ep_shard_buffers(ep_sim *sim, void **send_dptr, void **recv_dptr);
int ep_halo_pack(ep_sim *sim);
int ep_halo_unpack(ep_sim *sim);
int ep_halo_exchange_local(ep_sim **sims, int n_parts);

/* Choose the cell model and set every cell to an initial state.
 *   cell_type [n_tets] TP06: 0 endo, 1 mid, 2 epi (reading B5); NULL => 0
 *   y0        [n_types*S] one state vector per cell type (n_types = 3 for TP06, 1 for CRN98 and STEWART); NULL => built-in
 *             rest state (Stewart: the published initial state, a point of its spontaneous cycle -- the model has no rest)
 * Resets the step counter, the activation times (to -1) and keeps the stimulus slots. */
int ep_state_init(ep_sim *sim, int model, const uint8_t *cell_type, const double *y0);

/* Stimulus of eq. (4): I_s = amplitude on the listed cells while t_start <= t < t_start+duration,
 * with the window taken on integer step indices (reading A16).  amplitude in uA/cm^2; NEGATIVE depolarises (A15).
 * slot in [0, EP_MAX_STIM_SLOTS); n_cells = 0 clears the slot.  Overlapping slots add. */
int ep_stimulus_set(ep_sim *sim, int slot, int64_t n_cells, const int64_t *cell_ids, double amplitude_uA_cm2,
                    double t_start_ms, double duration_ms);

/* Triggered stimulus = the paper's communication-node coupling inside one mesh: the first time any of
 * the monitored cells exceeds 0 mV (threshold of PAPER.md:190), stimulus slot `slot` -- its cells, amplitude and duration
 * as given to ep_stimulus_set, its own t_start ignored -- switches on delay_ms later (PAPER.md:196 uses 5 ms / 3 ms) for
 * its duration, on integer steps: steps n_fire + ceil(delay/dt) <= n < ... + ceil(duration/dt), n_fire = index after the
 * crossing step.  A trigger fires once; ep_state_init re-arms it.  trigger in [0, 4); n_monitor = 0 removes it.
 * A slot can be driven by one trigger only.  slot = -1: monitor only -- the trigger records its firing time and drives no
 * slot of this mesh (the coupling then goes to another handle through ep_couple). */
int ep_trigger_set(ep_sim *sim, int trigger, int64_t n_monitor, const int64_t *monitor_ids, int slot, double delay_ms);
/* Time (ms) at which the trigger fired = (crossing step + 1) * dt, or -1.  Synchronises. */
int ep_trigger_time(ep_sim *sim, int trigger, double *t_fire_ms);

/* Communication-node coupling ACROSS two handles (the 2D Purkinje sheet excites the 3D ventricular
 * myocardium through the Purkinje-muscle junctions with an orthodromic delay of 5 ms; the bundles excite the
 * atria; with the roles exchanged the same call gives the antidromic direction).  If trigger `trigger` of
 * `src` has fired at t_f, stimulus slot `slot` of `dst` -- cells, amplitude and duration as given to ep_stimulus_set, e.g.
 * the cells within R_S of the junction -- is scheduled to switch on at t_f + delay_ms; *scheduled = 1 from then on, 0 before.
 * Call it between ep_step calls, both handles at the same time level, at intervals no longer than delay_ms: the trigger time
 * is read from the device (synchronises src), the window is resolved on dst's integer steps (reading A16).
 * EP_ERR_STATE if dst has already passed t_f + delay_ms (polled too late) or its slot has no cells. */
int ep_couple(ep_sim *src, int trigger, ep_sim *dst, int slot, double delay_ms, int *scheduled);

/* Advance n_steps explicit steps of size dt_ms (everything on the right-hand side at t^n; gates by
 * Rush-Larsen, the rest by forward Euler; v by eq. (7)).  Asynchronous on the sim's stream; errors are sticky.
 * EP_ERR_STATE: before ep_state_init, dt <= 0, or dt different from the previous call's after the first step. */
int ep_step(ep_sim *sim, int64_t n_steps, double dt_ms);

/* Order of the time stepping.  1 (default): the paper's scheme, Rush-Larsen gates + forward Euler.
 * 2: the improvement PAPER.md:232 names -- second-order Adams-Bashforth for v and the concentrations, and a second-order
 * Rush-Larsen step for the gates (steady state and time constant taken at arguments extrapolated to t^{n+1/2}; DESIGN.md
 * reading H1); the stimulus, piecewise constant on steps, is integrated exactly.  TP06 only (EP_ERR_ARG otherwise).  The first
 * step after ep_state_init / ep_write_state(s) / this call has no history and is a first-order step.  The explicit stability
 * limit of the diffusion part halves (AB2: dt <= chi Cm / rho(A), half of what ep_stable_dt reports).  Eight more state
 * rows per cell are read and written (64 + 64 B).  The history is not part of a checkpoint: a resumed run restarts with one
 * first-order step. */
int ep_set_time_order(ep_sim *sim, int order);

/* Wait for all queued work of this sim; returns the sticky error if any (EP_ERR_NUMERIC if a non-finite Vm was seen by
 * ep_check_finite). */
int ep_synchronize(ep_sim *sim);

/* Read-back, caller's cell order; each synchronises. */
int ep_read_vm(ep_sim *sim, double *out /*[n_tets]*/);
int ep_read_state(ep_sim *sim, int var /*0..S-1, 0 = Vm*/, double *out /*[n_tets]*/);
int ep_write_state(ep_sim *sim, int var, const double *in /*[n_tets]*/);
/* All S state rows in one call, row-major [S][n_tets] in the caller's cell order (row 0 = Vm).  The rows move through a
 * two-slot device staging buffer: the host<->device copy of row k overlaps the permutation kernel of row k-1 on a second
 * stream, and the host is synchronised once, at the end.  Pinned host memory makes the copies asynchronous. */
int ep_write_states(ep_sim *sim, const double *in /*[S*n_tets]*/);
int ep_read_states(ep_sim *sim, double *out /*[S*n_tets]*/);
/* First instant Vm exceeded 0 mV (reading A18: t=(n+1)dt of the step that crossed); -1 where never. */
int ep_activation_times(ep_sim *sim, double *out /*[n_tets]*/);

/* Checkpoint / resume.  A run is the S state rows (ep_read_states) PLUS the clock, the activation times recorded so far
 * and the firing state of the triggers; stimulus windows and trigger delays are counted on the integer step index
 * (readings A16, A17), so a resumed run needs that index back.  Restore order: ep_state_init, ep_stimulus_set /
 * ep_trigger_set as in the original run, ep_write_states, ep_set_step_count, ep_write_activation_times,
 * ep_trigger_restore.  The continuation is then bit-identical to the uninterrupted run.
 *   ep_set_step_count: step counter n (t = n dt) and the dt the run uses; ep_step keeps refusing any other dt.
 *   ep_write_activation_times: [n_tets], -1 where not yet activated (what ep_activation_times returned).
 *   ep_trigger_restore: the value ep_trigger_time returned (-1: not fired yet). */
int ep_set_step_count(ep_sim *sim, int64_t step_count, double dt_ms);
int ep_write_activation_times(ep_sim *sim, const double *in /*[n_tets]*/);
int ep_trigger_restore(ep_sim *sim, int trigger, double t_fire_ms);

/* Volume-averaged potential v_bar = sum_c V_c v_c / sum_c V_c at the current time (the paper's
 * convergence observable).  Deterministic two-pass reduction on the device; synchronises. */
int ep_mean_vm(ep_sim *sim, double *vbar_mV);

/* Diagnostics.  D = div(M grad v) in uA/cm^3 for a host cell field v [mV], through the device gather tables. */
int ep_apply_diffusion(ep_sim *sim, const double *v /*[n_tets]*/, double *D /*[n_tets]*/);
/* Largest explicit step of the diffusion part alone: 2 chi Cm / rho(A), rho by power iteration on the device. */
int ep_stable_dt(ep_sim *sim, double *dt_max_ms);
/* Scans Vm and every state row: sets *all_finite = 0 and the sticky error EP_ERR_NUMERIC if any value is NaN/Inf or any
 * ion concentration is <= 0 (forward Euler at an unstable dt; the kernels' logarithms need positive arguments and their
 * clamps would otherwise keep producing finite, meaningless numbers).  Synchronises. */
int ep_check_finite(ep_sim *sim, int *all_finite);

/* Stream interop: cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL => the sim's own stream. */
int ep_set_stream(ep_sim *sim, void *cuda_stream);
/* Zero-copy DEVICE views, valid until the next ep_step/ep_state_init: *vm_dptr -> double[n_tets] current Vm in device
 * (permuted) order, *perm_dptr -> int32[n_tets] with perm[device index] = caller's cell id.  Either may be NULL. */
int ep_device_vm(ep_sim *sim, void **vm_dptr, void **perm_dptr);

int64_t ep_n_cells(const ep_sim *sim);
int64_t ep_n_nodes(const ep_sim *sim);
int64_t ep_step_count(const ep_sim *sim);
double ep_time(const ep_sim *sim); /* step_count * dt (reading A17) */
/* Device bytes held by the sim, and the algorithmic HBM bytes one time step must move. */
int64_t ep_device_bytes(const ep_sim *sim);
int64_t ep_step_bytes(const ep_sim *sim);
/* Kernel launches issued by this sim so far (bench.py's gpu_launches). */
int64_t ep_launch_count(const ep_sim *sim);
/* Algorithmic HBM bytes of ONE launch of a step kernel: kernel 0 = node gather (S1), 1 = fused cell step (S2..S9). */
int64_t ep_kernel_bytes(const ep_sim *sim, int kernel);
/* Per-kernel device timing of ep_step with CUDA events on the sim's stream (for the roofline figures).
 * ep_profile(sim, 1) starts bracketing every step-kernel launch with an event pair and resets the totals;
 * ep_profile(sim, 0) stops.  ep_profile_read synchronises and returns the totals since the last reset:
 * out4 = { number of steps timed, total ms in kernel 0, total ms in kernel 1, 0 }. */
int ep_profile(ep_sim *sim, int enable);
int ep_profile_read(ep_sim *sim, double *out4);
void ep_destroy(ep_sim *sim);
const char *ep_last_error(void);

/* Diagnostic: evaluate one of the kernels' fp64 math routines (csrc/ep_math.cuh) on the device, element by element.
 * fn 0: 2^x (|x| <= 1000; the kernels form every exponent in base-2 units), 1: log (x positive, normal), 2: reciprocal,
 * 3: reciprocal square root.  Host pointers. */
int ep_math_eval(int fn, int64_t n, const double *x, double *y);

/* Diagnostic: measured throughput of the plain fp64 pipe of the current device, in warp-wide DFMA instructions per second
 * (a DFMA-only kernel, four independent chains per thread, 16 warps per SM sub-partition, best of three ~2 ms launches on
 * the default stream).  This is the denominator of the "alu" roof of DESIGN.md section 6: the fused step executes a
 * counted number of fp64 warp instructions per 32 cells (t_roof = max(bytes/BW_HBM, I_alg/R_fp64)). */
int ep_fp64_rate(double *warp_dfma_per_s);

/* The one call that allocates nothing -- for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid it); every other call works on a handle whose buffers ep_mesh_create allocated.
 * Weighted mean of a caller-owned DEVICE array: out_dev[0] = sum_i w_i v_i / sum_i w_i, out_dev[1] = sum_i w_i; with
 * v = the potentials of ep_device_vm() and w = the cell volumes in the same order this is the volume-averaged potential
 * v_bar of PAPER.md:216 / :230 that ep_mean_vm returns (a variant of its deterministic two-pass reduction; the summation
 * order differs, so the two agree to rounding, ~1e-13 relative, not bit for bit).
 *   v_dev, w_dev  DEVICE pointers, double[n], read only          out_dev  DEVICE pointer, double[2], written
 *   cuda_stream   cudaStream_t the two kernels are launched on (NULL: the default stream).  The call does NOT synchronise:
 *                 out_dev is valid once the stream has reached this point.
 * Scratch: a file-scope device array of 128 KB (one partial sum of w v and of w per 4,096 elements) that every GPU which
 * loads the library holds until the process exits; hence n <= EP_NOALLOC_MAX_N, larger n is refused with EP_ERR_ARG and a
 * message that names the limit.  No cudaMalloc / cudaFree / allocating library routine is called; the first call on each
 * device resolves the array's device address (cudaGetSymbolAddress, no allocation; make that call before capturing).
 * All calls share the array and it keeps the last call's contents (nothing in it needs to start at zero: each call reads
 * only the slots it has just written).  Calls that OVERLAP on the GPU -- different streams, concurrent graph replays --
 * race on it; calls ordered on one stream do not.  Runs on the current device; the pointers must belong to it.
 * Errors: EP_ERR_ARG (NULL pointer, n <= 0, n > EP_NOALLOC_MAX_N), EP_ERR_CUDA. */
#define EP_NOALLOC_MAX_N 33554432LL /* 8,192 blocks x 4,096 elements */
int ep_weighted_mean_noalloc(const double *v_dev, const double *w_dev, int64_t n, double *out_dev, void *cuda_stream);

/* Host-only preprocessor output for tests (no CUDA call is made).  Returns the factored stencil in the CALLER's
 * numbering: for cell c,  dv_diff[c] = sum_{m<8} a[c*8+m] * v_node[node[c*8+m]] + sum_{j<4} b[c*4+j] * (v[nbr[c*4+j]] - v[c])
 * in mV/ms (= D_c/(chi Cm)), where v_node[n] = sum_{k<node_deg[n]} w[node_ptr[n]+k] * v[node_cell[node_ptr[n]+k]].
 * Unused slots have coefficient 0 and a valid index.  Caller-allocated: node [n_tets*8] int32, a [n_tets*8],
 * nbr [n_tets*4] int32, b [n_tets*4], node_ptr [n_nodes+1] int64, node_cell/w [n_tets*4]; perm [n_tets] int32 (device
 * position -> caller cell id).  Any output pointer may be NULL. */
int ep_host_stencil(int64_t n_nodes, const double *xyz_mm, int64_t n_tets, const int32_t *tets, const double *fibre,
                    const double *sigma_scale, double sigma_l, double sigma_t, double chi, double Cm, int32_t *node,
                    double *a, int32_t *nbr, double *b, int64_t *node_ptr, int32_t *node_cell, double *w,
                    int32_t *perm);

/* The same for a triangulated surface (ep_mesh_create_tri): node [n_tris*8] (3 own + up to 3 opposite nodes, rest unused),
 * nbr / b [n_tris*4] (slot 3 unused), node_cell / w [n_tris*3]. */
int ep_host_stencil_tri(int64_t n_nodes, const double *xyz_mm, int64_t n_tris, const int32_t *tris, const double *fibre,
                        const double *sigma_scale, double sigma_l, double sigma_t, double chi, double Cm, int32_t *node,
                        double *a, int32_t *nbr, double *b, int64_t *node_ptr, int32_t *node_cell, double *w,
                        int32_t *perm);

#ifdef __cplusplus
}
#endif
#endif /* EP_H_ */
