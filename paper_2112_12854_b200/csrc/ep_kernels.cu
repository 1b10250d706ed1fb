// ep_kernels.cu -- sm_100a kernels of the monodomain + cell-model step.  fp64 throughout.
//
// Layout: cells and nodes are in Morton order; consecutive threads always touch consecutive
// addresses (coalesced 8-byte loads/stores); arrays with several rows per cell (state, stencil tables) are tile-major:
// the rows of the 128 cells of one thread block are contiguous, so each row is at a compile-time offset from one
// pointer.  The stencil is a fixed-width gather (8 node + 4 neighbour coefficients per cell, sliced-ELL node table), so
// the diffusion term needs no atomics and the result is deterministic (the only atomic is the once-per-run firing of a
// communication-node trigger).  Nothing here is a dense contraction: no tensor cores.
#include "ep_kernels.cuh"
#include <algorithm>
#include "ep_tp06.cuh"
#include "ep_crn98.cuh"
#include "ep_stewart.cuh"

namespace epk {

namespace {

// Programmatic dependent launch (PDL): the two step kernels are launched with programmatic stream serialisation, so the
// next kernel's blocks may start while the previous kernel drains its last wave.  pdl_wait() blocks until the previous
// kernel has completed and its writes are visible; pdl_launch_dependents() lets the next kernel in the stream start its
// prologue.  Both are no-ops for a kernel launched without the attribute.  Order of the chain cell(n-1) -> node(n) ->
// cell(n): node(n) waits first and only then releases cell(n), so cell(n) may read everything cell(n-1) wrote (state rows,
// Vm) as soon as it starts; it waits only before it touches the node values v_n that node(n) is still writing.  cell(n)
// releases node(n+1) at once: that kernel reads nothing but its slice pointers before its own wait, and it overwrites v_n
// only after cell(n) has completed.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

constexpr int CELL_THREADS = 128;   // = the tile of the tile-major layout
__host__ __device__ inline int64_t tile_index(int64_t i, int64_t k, int64_t rows) {
    return ((i / CELL_THREADS) * rows + k) * CELL_THREADS + i % CELL_THREADS;
}
constexpr int NODE_THREADS = 256;

// ---------------------------------------------------------------------------------------------------------
// S1: cell -> node interpolation.  A slice of 32 nodes is stored [k][lane]; NODE_PARTS warps share a slice, warp p
// takes rows k = p, p + NODE_PARTS, ... (each row read is 32 consecutive entries: fully coalesced) and the partial sums
// meet in shared memory.  Four times the threads of a warp-per-slice mapping; the kernel is a dependent gather (index,
// then value) that runs at 64 % of the HBM peak (profiles/r01b_to_r01e_cell_kernel.md, node kernel section).
// Resident blocks per SM the node kernel is compiled for: 6 (40 registers, 48 warps).  Measured on config 3 with six table rows
// in flight per warp: 67 registers 43.0 us, 59 registers 36.7 us, 40 registers 31.7 us, 32 registers (8 blocks) 34.3 us.
#ifndef EP_NODE_MIN_BLOCKS
#define EP_NODE_MIN_BLOCKS 6
#endif
constexpr int NODE_PARTS = 4;
constexpr int NODE_SLICES_PER_BLOCK = NODE_THREADS / 32 / NODE_PARTS;
__global__ void __launch_bounds__(NODE_THREADS, EP_NODE_MIN_BLOCKS) node_gather_kernel(int64_t nn, int64_t n_slices,
                                                                    const int64_t* __restrict__ slice_ptr,
                                                                    const int32_t* __restrict__ nidx,
                                                                    const double* __restrict__ nw,
                                                                    const double* __restrict__ vm,
                                                                    double* __restrict__ vn) {
    __shared__ double part[NODE_SLICES_PER_BLOCK][NODE_PARTS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sl = warp / NODE_PARTS, p = warp % NODE_PARTS;
    const int64_t slice = (int64_t)blockIdx.x * NODE_SLICES_PER_BLOCK + sl;
    double acc0 = 0.0, acc1 = 0.0;
    int64_t beg = 0, end = 0;
    if (slice < n_slices) { beg = __ldg(slice_ptr + slice); end = __ldg(slice_ptr + slice + 1); }
    pdl_wait();                  // Vm of this time level is complete (previous cell kernel); v_n is free to overwrite
    pdl_launch_dependents();     // the cell kernel may start its state loads now
    if (slice < n_slices) {
        int64_t q = beg + 32 * p + lane;
        const int64_t step = 32 * NODE_PARTS;
#ifndef EP_NODE_INFLIGHT
#define EP_NODE_INFLIGHT 6
#endif
        constexpr int NF = EP_NODE_INFLIGHT;      // rows of this warp in flight per trip: NF table loads, then NF dependent gathers
        for (; q < end; q += NF * step) {
            int32_t ii[NF];
            double ww[NF], vv[NF];
#pragma unroll
            for (int r = 0; r < NF; ++r) {
                const bool on = q + r * step < end;
                ii[r] = 0; ww[r] = 0.0;
                if (on) { ii[r] = ep_ldg_stream(nidx + q + r * step); ww[r] = ep_ldg_stream(nw + q + r * step); }
            }
#pragma unroll
            for (int r = 0; r < NF; ++r) vv[r] = vm[ii[r]];   // padded rows: weight 0 times vm[0]
#pragma unroll
            for (int r = 0; r < NF; ++r) {
                if (r & 1) acc1 = fma(ww[r], vv[r], acc1);
                else acc0 = fma(ww[r], vv[r], acc0);
            }
        }
    }
    part[sl][p][lane] = acc0 + acc1;
    __syncthreads();
    if (p == 0 && slice < n_slices) {
        const int64_t n = slice * 32 + lane;
        if (n < nn) vn[n] = (part[sl][0][lane] + part[sl][1][lane]) + (part[sl][2][lane] + part[sl][3][lane]);
    }
}

// S2+S3: the factored diffusion gather.  dv = sum_m a_m v_n[node_m] + sum_j b_j (v[nbr_j] - v_c)   [mV/ms]
__device__ __forceinline__ double diffusion_gather(int64_t i, const int32_t* __restrict__ cidx,
                                                   const double* __restrict__ ccoef, const double* __restrict__ vm,
                                                   const double* __restrict__ vn, double vc) {
    int32_t id[12];
    double cf[12];
#pragma unroll
    for (int m = 0; m < 12; ++m) {
        id[m] = __ldg(cidx + tile_index(i, m, 12));
        cf[m] = __ldg(ccoef + tile_index(i, m, 12));
    }
    double accn = 0.0, accc = 0.0;
#pragma unroll
    for (int m = 0; m < 8; ++m) accn = fma(cf[m], vn[id[m]], accn);
#pragma unroll
    for (int j = 0; j < 4; ++j) accc = fma(cf[8 + j], vm[id[8 + j]] - vc, accc);
    return accn + accc;
}

__global__ void __launch_bounds__(CELL_THREADS) diffusion_only_kernel(int64_t nc,
                                                                      const int32_t* __restrict__ cidx,
                                                                      const double* __restrict__ ccoef,
                                                                      const double* __restrict__ vm,
                                                                      const double* __restrict__ vn,
                                                                      double* __restrict__ out,
                                                                      const double* __restrict__ vol, double scale) {
    const int64_t i = (int64_t)blockIdx.x * CELL_THREADS + threadIdx.x;
    if (i >= nc) return;
    const double d = diffusion_gather(i, cidx, ccoef, vm, vn, vm[i]);
    out[i] = scale * (vol ? vol[i] * d : d);
}

// S2..S9 fused.  One thread per cell; state rows are read once and written once.  MODEL 0: TP06, 1: Courtemanche,
// 2: Stewart (Purkinje).
#ifndef EP_CELL_MIN_BLOCKS
#define EP_CELL_MIN_BLOCKS 4
#endif
template <int MODEL, int ORDER = 1>
__global__ void __launch_bounds__(CELL_THREADS, EP_CELL_MIN_BLOCKS) cell_step_kernel(int64_t nc,
                                                                                     const int32_t* __restrict__ cidx,
                                                                                     const double* __restrict__ ccoef,
                                                                                     StepArgs a) {
    // per-thread columns of the slot array (parked gate values of the cell models): slot s of thread t at xs[s][t]
    constexpr bool CF_SMEM = false;   // stencil coefficients in registers: with the streaming cell models shared-memory traffic costs
                                      // more than the 24 registers do (178.0 vs 179.6 us on config 3; the opposite held in round 1)
    constexpr int MSLOTS = (MODEL == 0) ? tp06::N_SLOTS : (MODEL == 1 ? crn::N_SLOTS : stw::N_SLOTS);
    constexpr int NSLOTS = MSLOTS + (CF_SMEM ? 12 : 0);
    __shared__ double xs[NSLOTS][CELL_THREADS];
    const int64_t i = (int64_t)blockIdx.x * CELL_THREADS + threadIdx.x;
    pdl_launch_dependents();
    if (i >= nc) return;
    const double v_old = a.vm_cur[i];
    // tile-major tables: every row of this block's tile is at a compile-time offset from these three pointers
    constexpr int S = (MODEL == 0) ? (int)TP06_S : (MODEL == 1 ? (int)CRN_S : (int)STW_S);
    const int32_t* tidx = cidx + (int64_t)blockIdx.x * (12 * CELL_THREADS) + threadIdx.x;
    const double* tcoef = ccoef + (int64_t)blockIdx.x * (12 * CELL_THREADS) + threadIdx.x;
    double* ycol = a.y + (int64_t)blockIdx.x * (S * CELL_THREADS) + threadIdx.x;
    static_assert(NSLOTS * CELL_THREADS * 8 <= 48 * 1024, "static shared memory limit");
    // S2+S3 in two halves: indices and coefficients are loaded here, the gathers are issued once the cell model has
    // parked its gates and stay in flight while it evaluates its logarithms and first exponential batch
    int32_t id[12];
    double cf[12];
#pragma unroll
    for (int m = 0; m < 12; ++m) {
        id[m] = ep_ldg_stream(tidx + m * CELL_THREADS);
        if constexpr (CF_SMEM) ep_cp_async8(&xs[MSLOTS + m][threadIdx.x], tcoef + m * CELL_THREADS);
        else cf[m] = ep_ldg_stream(tcoef + m * CELL_THREADS);
    }
    double gv[12];
    auto issue_gather = [&]() {
#pragma unroll
        for (int j = 0; j < 4; ++j) gv[8 + j] = a.vm_cur[id[8 + j]];
        pdl_wait();              // the node kernel of this step has finished writing v_n
#pragma unroll
        for (int m = 0; m < 8; ++m) gv[m] = a.vn[id[m]];
    };
    auto finish_gather = [&]() {   // dv = sum_m a_m v_n[node_m] + sum_j b_j (v[nbr_j] - v_c)   [mV/ms]
        double accn = 0.0, accm = 0.0, accc = 0.0;
        if constexpr (CF_SMEM) {
            ep_cp_async_wait();
#pragma unroll
            for (int m = 0; m < 12; ++m) cf[m] = xs[MSLOTS + m][threadIdx.x];
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            accn = fma(cf[m], gv[m], accn);
            accm = fma(cf[4 + m], gv[4 + m], accm);
            accc = fma(cf[8 + m], gv[8 + m] - v_old, accc);
        }
        const double dv = (accn + accm) + accc;
        return a.dv_extra ? dv + a.dv_extra[i] : dv;     // bidomain: + div(M_int grad v_ext)/(chi C_m), eq. (1)
    };
    // S4: stimulus, eq. (4) PAPER.md:130-132 (window already resolved on the host into istim[k]).  The mask is requested
    // here with the other loads; the cell model calls stimulus() after its first exponential batch, so nothing waits for it.
    const unsigned mask = a.smask[i];
    auto stimulus = [&]() {
        double istim = 0.0;
        if (mask != 0) {   // few cells belong to a stimulus slot: one test instead of eight for the others
            const long long n = a.desc ? a.desc->n : a.inl.n;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (!(mask & (1u << k))) continue;
                if (a.trig_slots & (1u << k)) {
                    // slot driven by a trigger: on for ndur steps starting nd steps after the monitored crossing.  A firing
                    // written by another thread of THIS launch cannot switch it on (n_on >= n + 1), so there is no race.
                    for (int t = 0; t < MAX_TRIGGERS; ++t) {
                        const TrigPar p = a.trig_par[t];
                        if (!p.armed || p.slot != k) continue;
                        const long long nf = a.trig_fire[t];
                        if (nf >= 0 && n >= nf + p.nd && n < nf + p.nd + p.ndur) istim += p.amp_cm;
                    }
                } else {
                    istim += a.desc ? a.desc->istim[k] : a.inl.istim[k];
                }
            }
        }
        return istim;
    };
    double v_new;
    if constexpr (MODEL == 0 && ORDER == 2) {
        O2Hist h;
        h.hcol = a.hist + (int64_t)blockIdx.x * (O2_ROWS * CELL_THREADS) + threadIdx.x;
        h.stride = CELL_THREADS;
        h.v_prev = a.vm_next[i];          // the buffer about to be overwritten still holds v^{n-1}
        h.have = a.o2_have;
        v_new = tp06_step<2, CELL_THREADS>(v_old, ycol, CELL_THREADS, a.ctype[i], a.dt, stimulus, issue_gather,
                                           finish_gather, &xs[0][threadIdx.x], h);
    } else if constexpr (MODEL == 0)
        v_new = tp06_step<1, CELL_THREADS>(v_old, ycol, CELL_THREADS, a.ctype[i], a.dt, stimulus, issue_gather, finish_gather,
                                           &xs[0][threadIdx.x]);
    else if constexpr (MODEL == 1)
        v_new = crn_step<CELL_THREADS>(v_old, ycol, CELL_THREADS, a.dt, stimulus, issue_gather, finish_gather,
                                       &xs[0][threadIdx.x]);
    else
        v_new = stw_step<CELL_THREADS>(v_old, ycol, CELL_THREADS, a.dt, stimulus, issue_gather, finish_gather,
                                       &xs[0][threadIdx.x]);
    a.vm_next[i] = v_new;
    // S9: activation time = first upward crossing of 0 mV (reading A18)
    if (v_old <= 0.0 && v_new > 0.0) {
        if (a.tact[i] < 0.0) a.tact[i] = a.desc ? a.desc->t_next : a.inl.t_next;
        // communication nodes: the first monitored cell to exceed 0 mV fires its trigger, once
        const unsigned tm = a.tmask[i];
        if (tm != 0) {
            const unsigned long long n1 = (unsigned long long)((a.desc ? a.desc->n : a.inl.n) + 1);
            for (int t = 0; t < MAX_TRIGGERS; ++t)
                if (tm & (1u << t)) atomicCAS((unsigned long long*)(a.trig_fire + t), ~0ull, n1);
        }
    }
}

__global__ void state_fill_kernel(int S, int64_t nc, int64_t nc_pad, const uint8_t* __restrict__ ctype,
                                  const double* __restrict__ y0, double* __restrict__ y, double* __restrict__ vm,
                                  double* __restrict__ tact) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nc_pad) return;
    const int t = (i < nc) ? ctype[i] : 0;
    for (int k = 0; k < S; ++k) {
        const double val = y0 ? y0[t * S + k]
                              : (S == (int)TP06_S ? TP06_REST_STATE[k] : (S == (int)CRN_S ? CRN_REST_STATE[k] : STW_INIT_STATE[k]));
        if (k == 0) vm[i] = val; else y[tile_index(i, k, S)] = val;
    }
    tact[i] = -1.0;
}

__global__ void gather_f64_kernel(int64_t n, const double* __restrict__ src, const int32_t* __restrict__ idx,
                                  double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[idx[i]];
}
__global__ void scatter_f64_kernel(int64_t n, const double* __restrict__ src, const int32_t* __restrict__ idx,
                                   double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[idx[i]] = src[i];
}
// state row k (tile-major, S rows) <-> a linear array in another numbering: dst[c] = y[(idx[c], k)] / y[(i, k)] = src[idx[i]]
__global__ void state_row_get_kernel(int64_t n, const double* __restrict__ y, int S, int k,
                                     const int32_t* __restrict__ idx, double* __restrict__ dst) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < n) dst[c] = y[tile_index(idx[c], k, S)];
}
__global__ void state_row_put_kernel(int64_t n, const double* __restrict__ src, const int32_t* __restrict__ idx, int S,
                                     int k, double* __restrict__ y) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[tile_index(i, k, S)] = src[idx[i]];
}

// deterministic two-pass reductions: 1024 blocks x 256 threads, fixed tree
template <int MODE>   // 0: sum of squares, 1: count of non-finite entries, 2: sum of w[i] * x[i]
__global__ void __launch_bounds__(256) reduce_partial_kernel(int64_t n, const double* __restrict__ x,
                                                              const double* __restrict__ w,
                                                              double* __restrict__ partial) {
    __shared__ double sh[256];
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
        const double v = x[i];
        acc += (MODE == 0) ? v * v : (MODE == 1 ? (isfinite(v) ? 0.0 : 1.0) : w[i] * v);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void __launch_bounds__(1024) reduce_final_kernel(const double* __restrict__ partial, double* out) {
    __shared__ double sh[1024];
    sh[threadIdx.x] = partial[threadIdx.x];
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = sh[0];
}
// Failure detection over the WHOLE state (not only Vm): counts[0] += non-finite entries of Vm and of state rows 1..S-1,
// counts[1] += concentrations (rows conc0..S-1) that are not positive -- forward Euler at an unstable dt can drive them
// through zero, after which the logarithms of the reversal potentials mean nothing.  Integer counts: atomics are exact.
__global__ void __launch_bounds__(256) state_scan_kernel(int S, int conc0, int64_t nc, const double* __restrict__ vm,
                                                          const double* __restrict__ y,
                                                          unsigned long long* __restrict__ counts) {
    unsigned bad = 0, nonpos = 0;
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < nc; i += (int64_t)gridDim.x * 256) {
        bad += !isfinite(vm[i]);
        for (int k = 1; k < S; ++k) {
            const double v = y[tile_index(i, k, S)];
            bad += !isfinite(v);
            if (k >= conc0) nonpos += !(v > 0.0);
        }
    }
    bad = __reduce_add_sync(0xffffffffu, bad);
    nonpos = __reduce_add_sync(0xffffffffu, nonpos);
    if ((threadIdx.x & 31) == 0) {
        if (bad) atomicAdd(counts, (unsigned long long)bad);
        if (nonpos) atomicAdd(counts + 1, (unsigned long long)nonpos);
    }
}

__global__ void scale_by_inv_norm_kernel(int64_t n, const double* __restrict__ x, const double* __restrict__ norm2,
                                         double* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = x[i] / sqrt(norm2[0]);
}

__global__ void math_eval_kernel(int fn, int64_t n, const double* __restrict__ x, double* __restrict__ y) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double v[1] = {x[i]};
    if (fn == 0) ep_exp2_wide<1>(v);
    else if (fn == 1) ep_log_wide<1>(v);
    else if (fn == 2) v[0] = ep_rcp(v[0]);
    else v[0] = ep_rsqrt(v[0]);
    y[i] = v[0];
}

// Plain fp64-pipe throughput probe (the "alu" roof of DESIGN.md section 6): every thread runs `iters` x 8 x 4 DFMAs in four
// independent chains, 16 warps per SM sub-partition, no memory traffic.  Returns nothing useful in `out` (it only keeps
// the chains alive); the launcher times the kernel.
__global__ void __launch_bounds__(512) dfma_rate_kernel(double* out, int iters, double a, double b) {
    double x[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) x[j] = threadIdx.x * 1e-9 + j;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int j = 0; j < 4; ++j) x[j] = fma(x[j], a, b);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = (x[0] + x[1]) + (x[2] + x[3]);
}

inline unsigned blocks_for(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

}  // namespace

void launch_math_eval(int fn, int64_t n, const double* x, double* y, cudaStream_t s) {
    math_eval_kernel<<<blocks_for(n, 256), 256, 0, s>>>(fn, n, x, y);
}

double launch_dfma_rate(double* scratch, int64_t scratch_len, int iters, cudaStream_t s) {
    const int threads = 512;
    const unsigned blocks = (unsigned)std::min<int64_t>(592, scratch_len / threads);
    if (blocks == 0) return 0.0;
    dfma_rate_kernel<<<blocks, threads, 0, s>>>(scratch, iters, 0.999999, 1e-7);
    return (double)blocks * (threads / 32) * (double)iters * 32.0;   // warp-wide DFMAs issued
}

int model_n_states(int model) { return model == 0 ? (int)TP06_S : (model == 1 ? (int)CRN_S : (model == 2 ? (int)STW_S : -1)); }

// kernel launch with the programmatic-stream-serialisation attribute (see the PDL note at the top of this file)
template <class... KArgs, class... Args>
void launch_pdl(void (*kernel)(KArgs...), unsigned grid, unsigned block, cudaStream_t s, bool pdl, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

void launch_node_gather(const DeviceMesh& m, const double* vm, double* vn, cudaStream_t s, bool pdl) {
    const unsigned grid = blocks_for(m.n_slices, NODE_SLICES_PER_BLOCK);
    launch_pdl(node_gather_kernel, grid, NODE_THREADS, s, pdl, m.nn, m.n_slices, m.slice_ptr, m.nidx, m.nw, vm, vn);
}

void launch_cell_step(const DeviceMesh& m, int model, const StepArgs& a, cudaStream_t s, bool pdl) {
    const int64_t nact = m.nc_active > 0 ? m.nc_active : m.nc;
    const unsigned grid = blocks_for(nact, CELL_THREADS);
    if (model == 0 && a.hist) launch_pdl(cell_step_kernel<0, 2>, grid, CELL_THREADS, s, pdl, nact, m.cidx, m.ccoef, a);
    else if (model == 0) launch_pdl(cell_step_kernel<0>, grid, CELL_THREADS, s, pdl, nact, m.cidx, m.ccoef, a);
    else if (model == 1) launch_pdl(cell_step_kernel<1>, grid, CELL_THREADS, s, pdl, nact, m.cidx, m.ccoef, a);
    else launch_pdl(cell_step_kernel<2>, grid, CELL_THREADS, s, pdl, nact, m.cidx, m.ccoef, a);
}

void launch_diffusion_only(const DeviceMesh& m, const double* vm, const double* vn, double* out, cudaStream_t s,
                           const double* ccoef, const double* vol, double scale) {
    diffusion_only_kernel<<<blocks_for(m.nc, CELL_THREADS), CELL_THREADS, 0, s>>>(m.nc, m.cidx, ccoef ? ccoef : m.ccoef, vm,
                                                                                  vn, out, vol, scale);
}

void launch_state_fill(int model, int64_t nc, int64_t nc_pad, const uint8_t* ctype, const double* y0_dev, double* y,
                       double* vm, double* tact, cudaStream_t s) {
    state_fill_kernel<<<blocks_for(nc_pad, 256), 256, 0, s>>>(model_n_states(model), nc, nc_pad, ctype, y0_dev, y, vm,
                                                              tact);
}

void launch_scatter_f64(int64_t n, const double* src, const int32_t* idx, double* dst, cudaStream_t s) {
    if (n > 0) scatter_f64_kernel<<<blocks_for(n, 256), 256, 0, s>>>(n, src, idx, dst);
}
void launch_gather_f64(int64_t n, const double* src, const int32_t* idx, double* dst, cudaStream_t s) {
    gather_f64_kernel<<<blocks_for(n, 256), 256, 0, s>>>(n, src, idx, dst);
}
void launch_state_row_get(int64_t n, const double* y, int S, int k, const int32_t* inv, double* dst, cudaStream_t s) {
    state_row_get_kernel<<<blocks_for(n, 256), 256, 0, s>>>(n, y, S, k, inv, dst);
}
void launch_state_row_put(int64_t n, const double* src, const int32_t* perm, int S, int k, double* y, cudaStream_t s) {
    state_row_put_kernel<<<blocks_for(n, 256), 256, 0, s>>>(n, src, perm, S, k, y);
}
void launch_norm2(int64_t n, const double* x, double* partial, double* out, cudaStream_t s) {
    reduce_partial_kernel<0><<<1024, 256, 0, s>>>(n, x, nullptr, partial);
    reduce_final_kernel<<<1, 1024, 0, s>>>(partial, out);
}
void launch_count_nonfinite(int64_t n, const double* x, double* partial, double* out, cudaStream_t s) {
    reduce_partial_kernel<1><<<1024, 256, 0, s>>>(n, x, nullptr, partial);
    reduce_final_kernel<<<1, 1024, 0, s>>>(partial, out);
}
void launch_weighted_sum(int64_t n, const double* x, const double* w, double* partial, double* out, cudaStream_t s) {
    reduce_partial_kernel<2><<<1024, 256, 0, s>>>(n, x, w, partial);
    reduce_final_kernel<<<1, 1024, 0, s>>>(partial, out);
}
void launch_state_scan(int model, int64_t nc, const double* vm, const double* y, unsigned long long* counts,
                       cudaStream_t s) {
    const int S = model_n_states(model), conc0 = (model == 0) ? (int)Y_CAI : (model == 1 ? (int)C_NAI : (int)W_CAI);
    state_scan_kernel<<<1184, 256, 0, s>>>(S, conc0, nc, vm, y, counts);
}
void launch_scale_by_inv_norm(int64_t n, const double* x, const double* norm2, double* out, cudaStream_t s) {
    scale_by_inv_norm_kernel<<<blocks_for(n, 256), 256, 0, s>>>(n, x, norm2, out);
}

}  // namespace epk
