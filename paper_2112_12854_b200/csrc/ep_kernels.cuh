// ep_kernels.cuh -- launch interface between the C-ABI layer (ep_api.cu) and the sm_100a kernels (ep_kernels.cu).
#pragma once
#include <cstdint>
#include <functional>
#include <cuda_runtime.h>

namespace epk {

struct DeviceMesh {
    int64_t nc = 0, nn = 0, nc_pad = 0, n_slices = 0;
    int64_t nc_active = 0;              // cells the step kernel advances: nc, or the owned cells of a shard (they come first)
    const int32_t* cidx = nullptr;      // tile-major [nc_pad/128][12][128]
    const double* ccoef = nullptr;      // tile-major [nc_pad/128][12][128]
    const int64_t* slice_ptr = nullptr; // [n_slices+1]
    const int32_t* nidx = nullptr;
    const double* nw = nullptr;
};

// what changes from one time step to the next
// Triggered stimulus (communication-node coupling): host-written parameters of one trigger
struct TrigPar {
    int32_t armed;          // 0: unused
    int32_t slot;           // stimulus slot it drives
    int32_t nd, ndur;       // delay and duration in time steps
    double amp_cm;          // I_s / C_m of that slot
};
enum { MAX_TRIGGERS = 4 };
enum { O2_ROWS = 8 };     // history rows of the second-order scheme: f^{n-1} of v Ca_i Ca_SR Ca_SS Na_i K_i, Ca_SS^{n-1}, Ca_SR^{n-1}

struct StepDesc {
    long long n;            // step index
    double t_next;          // (n+1)*dt, recorded on an upward crossing of 0 mV
    double istim[8];        // I_s/C_m of each slot at step n (0 when the slot's window is closed)
};

struct StepArgs {
    const double* vm_cur;   // [nc_pad]
    double* vm_next;        // [nc_pad]
    double* y;              // tile-major [nc_pad/128][S][128]; row 0 unused (Vm lives in vm_cur/vm_next)
    double* vn;             // [nn] node values scratch
    const uint8_t* ctype;   // [nc_pad]
    const uint8_t* smask;   // [nc_pad] bit k = cell belongs to stimulus slot k
    double* tact;           // [nc_pad]
    const uint8_t* tmask;   // [nc_pad] bit t = cell is monitored by trigger t (read only on a 0 mV crossing)
    long long* trig_fire;   // [MAX_TRIGGERS] step index (n+1) of the first crossing of a monitored cell, -1 before
    const TrigPar* trig_par;// [MAX_TRIGGERS]
    unsigned trig_slots;    // bit k = slot k is driven by a trigger instead of its own time window
    double dt;
    double* hist;           // second-order stepping (TP06): tile-major [nc_pad/128][O2_ROWS][128] history of t^{n-1}, or NULL
    int o2_have;            // 0 on the first step after an initialisation (no history yet: first-order step)
    const double* dv_extra; // [nc_pad] extra right-hand side in mV/ms (bidomain: div(M_int grad v_ext)/(chi C_m)), or NULL
    const StepDesc* desc;   // device descriptor of this step (CUDA-graph replay), or NULL: use `inl`
    StepDesc inl;
};

// S1 of SURVEY 8(a): v_n = sum_k w_nk v_k
// pdl: launch with programmatic stream serialisation (the kernel's prologue may overlap the previous kernel's tail)
void launch_node_gather(const DeviceMesh& m, const double* vm, double* vn, cudaStream_t s, bool pdl = false);
// S2..S9 fused: diffusion gather + stimulus + cell model + RL/FE updates + Vm write + activation record
void launch_cell_step(const DeviceMesh& m, int model, const StepArgs& a, cudaStream_t s, bool pdl = false);
// out[i] = scale * (vol ? vol[i] : 1) * D_c/(chi Cm) [mV/ms] from vm and vn with the coefficient table `ccoef` (NULL: the mesh's
// own).  Diagnostics, and the operator applications of the bidomain solver.
void launch_diffusion_only(const DeviceMesh& m, const double* vm, const double* vn, double* out, cudaStream_t s,
                           const double* ccoef = nullptr, const double* vol = nullptr, double scale = 1.0);
// fill y rows with one state vector per cell type; y0 is a DEVICE pointer [n_types*S]; NULL = built-in rest state
void launch_state_fill(int model, int64_t nc, int64_t nc_pad, const uint8_t* ctype, const double* y0_dev, double* y,
                       double* vm, double* tact, cudaStream_t s);
// dst[idx[i]] = src[i] (halo unpack)
void launch_scatter_f64(int64_t n, const double* src, const int32_t* idx, double* dst, cudaStream_t s);
// permutation helpers: dst[i] = src[idx[i]]
void launch_gather_f64(int64_t n, const double* src, const int32_t* idx, double* dst, cudaStream_t s);
// state row k of the tile-major state array: dst[c] = y(inv[c], k)   /   y(i, k) = src[perm[i]]
void launch_state_row_get(int64_t n, const double* y, int S, int k, const int32_t* inv, double* dst, cudaStream_t s);
void launch_state_row_put(int64_t n, const double* src, const int32_t* perm, int S, int k, double* y, cudaStream_t s);
// reductions for the power iteration and the finite check (deterministic two-pass)
void launch_norm2(int64_t n, const double* x, double* partial /*[1024]*/, double* out /*[1]*/, cudaStream_t s);
void launch_scale_by_inv_norm(int64_t n, const double* x, const double* norm2, double* out, cudaStream_t s);
// out[0] = sum_i w[i] x[i], fixed summation tree (deterministic)
void launch_weighted_sum(int64_t n, const double* x, const double* w, double* partial, double* out, cudaStream_t s);
// counts[0] += non-finite entries of Vm and all state rows, counts[1] += non-positive concentrations (device, zeroed by caller)
void launch_state_scan(int model, int64_t nc, const double* vm, const double* y, unsigned long long* counts,
                       cudaStream_t s);
void launch_count_nonfinite(int64_t n, const double* x, double* partial, double* out, cudaStream_t s);

int model_n_states(int model);
// fp64-pipe probe: launches a DFMA-only kernel on up to 592 blocks x 512 threads (scratch must hold that many doubles),
// returns the number of warp-wide DFMAs it issues; the caller times it
double launch_dfma_rate(double* scratch, int64_t scratch_len, int iters, cudaStream_t s);
// diagnostics: y[i] = f(x[i]) with the kernels' own exp / log / rcp / rsqrt (device pointers)
void launch_math_eval(int fn, int64_t n, const double* x, double* y, cudaStream_t s);

// ---- restarted GMRES on the device (ep_elliptic.cu): bidomain elliptic equation
struct GmresOp {           // out = A x on stream s; `launches` = kernels one application issues
    std::function<void(const double*, double*, cudaStream_t)> f;
    int launches = 0;
    void operator()(const double* x, double* out, cudaStream_t s) const { f(x, out, s); }
};
struct Gmres {
    int m = 0;
    int64_t n = 0, stride = 0, bytes = 0;
    double *V = nullptr, *w = nullptr, *small = nullptr, *partial = nullptr;
    double *H = nullptr, *cs = nullptr, *sn = nullptr, *g = nullptr, *y = nullptr, *hcol = nullptr, *scal = nullptr;
};
int gmres_alloc(Gmres& G, int64_t n, int restart);      // 0, or negative on allocation failure / bad restart length
void gmres_free(Gmres& G);
// x: first estimate in, solution out.  Stops when the residual estimate <= rel_tol * |b|.  Returns the number of
// iterations, or a negative value on a CUDA error; *rel_res_out = last residual estimate / |b|.
// Also stops when the residual estimate <= abs_tol (a right-hand side that is round-off noise has no meaningful relative scale).
int gmres_solve(Gmres& G, const GmresOp& apply, const double* b, double* x, double rel_tol, double abs_tol, int max_cycles,
                int check_every, cudaStream_t s, double* rel_res_out, int64_t* launches);
// x <- 2 x - xprev (if have), xprev <- old x: linear extrapolation of the first estimate from the two previous solutions
void launch_extrapolate(int64_t n, double* x, double* xprev, int have, cudaStream_t s);
// x -= (sum_i x[i]) / n
void launch_remove_mean(const Gmres& G, double* x, cudaStream_t s);
// x -= (sum_i weight[i] x[i]) / total
void launch_remove_weighted_mean(const Gmres& G, double* x, const double* weight, double total, cudaStream_t s);

}  // namespace epk
