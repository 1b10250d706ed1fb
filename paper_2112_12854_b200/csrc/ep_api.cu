// ep_api.cu -- the C-ABI of include/ep.h: argument checks, host preprocessing, device memory, launches.
// There is no CPU fallback: every compute entry point needs a CUDA device and fails with EP_ERR_CUDA otherwise.
#include "../../include/ep.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "ep_host.h"
#include "ep_kernels.cuh"

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}

struct StimSlot {
    bool set = false;
    double amp = 0.0, t0 = 0.0, dur = 0.0;
    int64_t n_cells = 0;
};

}  // namespace

struct ep_sim {
    int64_t nc = 0, nn = 0, nc_pad = 0;
    double chi = 0.0, Cm = 0.0;
    // host copies kept for the life of the sim
    std::vector<int32_t> perm_c, inv_c;
    std::vector<uint8_t> smask_host;   // device order
    StimSlot stim[EP_MAX_STIM_SLOTS];
    int64_t star_entries = 0;
    // device
    epk::DeviceMesh dm;
    int32_t *d_cidx = nullptr, *d_nidx = nullptr, *d_perm = nullptr, *d_inv = nullptr;
    double *d_ccoef = nullptr, *d_nw = nullptr;
    int64_t* d_slice_ptr = nullptr;
    double *d_vm[2] = {nullptr, nullptr}, *d_y = nullptr, *d_vn = nullptr, *d_tact = nullptr, *d_tmp = nullptr,
           *d_tmp2 = nullptr, *d_red = nullptr;
    double* d_vol = nullptr;
    double vol_total = 0.0, vol_norm2 = 0.0;    // sum of the cell volumes, and their Euclidean norm
    uint8_t *d_ctype = nullptr, *d_smask = nullptr;
    int cur = 0;   // d_vm[cur] holds Vm at the current time level
    cudaStream_t own_stream = nullptr, stream = nullptr;
    int model = -1, S = 0;
    int64_t step = 0;
    double dt = 0.0;
    int sticky = EP_OK;
    int64_t dev_bytes = 0, launches = 0;
    // triggered stimuli (ep_trigger_set)
    struct Trig { bool armed = false; int slot = 0; double delay = 0.0; };
    Trig trig[epk::MAX_TRIGGERS];
    std::vector<uint8_t> tmask_host;   // device order
    uint8_t* d_tmask = nullptr;
    long long* d_trig_fire = nullptr;
    epk::TrigPar* d_trig_par = nullptr;
    bool trig_dirty = true;
    // CUDA-graph replay of GRAPH_STEPS time steps (launch-bound meshes), one graph per parity of the Vm double buffer;
    // rebuilt when dt, model or stream change
    cudaGraphExec_t graph[2] = {nullptr, nullptr};
    double graph_dt = 0.0;
    int graph_model = -1;
    cudaStream_t graph_stream = nullptr;
    int device = 0;                             // the device the handle was created on
    int dim = 3;                                // 3: tetrahedra, 2: triangulated surface
    // bidomain (ep_mesh_create_bidomain): the mesh's own tables hold M_int; second coefficient table for M_int + M_ext
    bool bidomain = false;
    double *d_ccoef_ie = nullptr, *d_vext = nullptr, *d_src = nullptr, *d_b = nullptr, *d_vext_prev = nullptr;
    int vext_hist = 0;                          // consecutive solutions held in d_vext / d_vext_prev (0, 1, 2)
    epk::Gmres gm;
    int bd_restart = 30, bd_max_cycles = 200, bd_check = 5;
    double bd_tol = 1e-10;
    bool vext_valid = false;
    // shard of a larger mesh (ep_shard_create): local cell k <-> global cell id, exchange lists as device positions
    int n_parts = 1, part = 0;
    int64_t n_owned = 0;
    std::vector<int64_t> shard_global, send_ptr, recv_ptr;
    int32_t *d_send_idx = nullptr, *d_recv_idx = nullptr;
    double *d_send = nullptr, *d_recv = nullptr;
    // second-order time stepping (ep_set_time_order): history rows and whether they hold t^{n-1} of the current state
    int order = 1;
    double* d_hist = nullptr;
    bool o2_have = false;
    int64_t bd_iters_last = 0, bd_iters_total = 0, bd_solves = 0;
    double bd_res_last = 0.0;
    bool pdl = true;                            // programmatic dependent launch of the step kernels (EP_NO_PDL=1 disables)
    // bulk state I/O (ep_write_states / ep_read_states): second stream + events for a two-slot staging pipeline
    cudaStream_t io_stream = nullptr;
    cudaEvent_t io_copied[2] = {}, io_consumed[2] = {}, io_fence = nullptr;
    epk::StepDesc* d_desc = nullptr;
    epk::StepDesc* h_desc = nullptr;            // pinned ring of DESC_RING x GRAPH_STEPS descriptors
    cudaEvent_t desc_ev[8] = {};                // copy-done events guarding the reuse of a ring slot
    bool desc_ev_used[8] = {};
    int desc_slot = 0;
    // per-kernel event timing (ep_profile)
    bool profiling = false;
    std::vector<cudaEvent_t> ev;       // 3 per step: before node kernel, between, after cell kernel
    size_t ev_used = 0;
    double prof_steps = 0.0, prof_ms[2] = {0.0, 0.0};
};

namespace {

#define EP_CUDA(sim, call)                                                                        \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess) {                                                                  \
            if (sim) (sim)->sticky = EP_ERR_CUDA;                                                 \
            return fail(e_ == cudaErrorMemoryAllocation ? EP_ERR_NOMEM : EP_ERR_CUDA,             \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                      \
        }                                                                                         \
    } while (0)

template <class T>
int dev_alloc(ep_sim* s, T** p, int64_t count) {
    const size_t bytes = (size_t)(count > 0 ? count : 1) * sizeof(T);
    EP_CUDA(s, cudaMalloc((void**)p, bytes));
    s->dev_bytes += (int64_t)bytes;
    return EP_OK;
}

template <class T>
int upload(ep_sim* s, T** p, const std::vector<T>& h) {
    int rc = dev_alloc(s, p, (int64_t)h.size());
    if (rc) return rc;
    if (!h.empty()) EP_CUDA(s, cudaMemcpy(*p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    return EP_OK;
}

int64_t step_index(double t, double dt) { return (int64_t)std::ceil(t / dt - 1e-9); }   // reading A16

void free_all(ep_sim* s) {
    void* ptrs[] = {s->d_cidx, s->d_nidx, s->d_perm, s->d_inv, s->d_ccoef, s->d_nw, s->d_slice_ptr, s->d_vm[0],
                    s->d_vm[1], s->d_y, s->d_vn, s->d_tact, s->d_tmp, s->d_tmp2, s->d_red, s->d_ctype, s->d_smask,
                    s->d_vol, s->d_tmask, s->d_trig_fire, s->d_trig_par, s->d_ccoef_ie, s->d_vext, s->d_src, s->d_b, s->d_hist, s->d_send_idx, s->d_recv_idx,
                    s->d_send, s->d_recv, s->d_vext_prev};
    epk::gmres_free(s->gm);
    for (void* p : ptrs) if (p) cudaFree(p);
    for (cudaEvent_t e : s->ev) cudaEventDestroy(e);
    for (cudaGraphExec_t g : s->graph) if (g) cudaGraphExecDestroy(g);
    if (s->d_desc) cudaFree(s->d_desc);
    for (int k = 0; k < 2; ++k) {
        if (s->io_copied[k]) cudaEventDestroy(s->io_copied[k]);
        if (s->io_consumed[k]) cudaEventDestroy(s->io_consumed[k]);
    }
    if (s->io_fence) cudaEventDestroy(s->io_fence);
    if (s->io_stream) cudaStreamDestroy(s->io_stream);
    if (s->h_desc) cudaFreeHost(s->h_desc);
    for (cudaEvent_t e : s->desc_ev) if (e) cudaEventDestroy(e);
    if (s->own_stream) cudaStreamDestroy(s->own_stream);
}

// fold the recorded event triples into the totals (synchronises)
int profile_drain(ep_sim* s) {
    if (s->ev_used == 0) return EP_OK;
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    for (size_t i = 0; i + 2 < s->ev_used; i += 3) {
        float a = 0.f, b = 0.f;
        EP_CUDA(s, cudaEventElapsedTime(&a, s->ev[i], s->ev[i + 1]));
        EP_CUDA(s, cudaEventElapsedTime(&b, s->ev[i + 1], s->ev[i + 2]));
        s->prof_ms[0] += a; s->prof_ms[1] += b; s->prof_steps += 1.0;
    }
    s->ev_used = 0;
    return EP_OK;
}

int profile_event(ep_sim* s) {
    if (s->ev_used == s->ev.size()) {
        cudaEvent_t e;
        EP_CUDA(s, cudaEventCreate(&e));
        s->ev.push_back(e);
    }
    EP_CUDA(s, cudaEventRecord(s->ev[s->ev_used++], s->stream));
    return EP_OK;
}

constexpr int GRAPH_STEPS = 32;   // even, so that the Vm double buffer is back where it started
constexpr int DESC_RING = 8;

void fill_desc(const ep_sim* s, int64_t n, double dt, const int64_t* n_on, const int64_t* n_off, epk::StepDesc& d) {
    d.n = n;
    d.t_next = (double)(n + 1) * dt;   // reading A17: time from the integer counter
    for (int k = 0; k < EP_MAX_STIM_SLOTS; ++k)
        d.istim[k] = (s->stim[k].set && n_on[k] <= n && n < n_off[k]) ? s->stim[k].amp / s->Cm : 0.0;
}

epk::StepArgs step_args(ep_sim* s, int cur, double dt) {
    epk::StepArgs a;
    a.vm_cur = s->d_vm[cur]; a.vm_next = s->d_vm[cur ^ 1];
    a.y = s->d_y; a.vn = s->d_vn; a.ctype = s->d_ctype; a.smask = s->d_smask; a.tact = s->d_tact;
    a.tmask = s->d_tmask; a.trig_fire = s->d_trig_fire; a.trig_par = s->d_trig_par;
    a.trig_slots = 0;
    for (const ep_sim::Trig& t : s->trig) if (t.armed && t.slot >= 0) a.trig_slots |= 1u << t.slot;
    a.dt = dt; a.desc = nullptr;
    a.dv_extra = s->bidomain ? s->d_src : nullptr;
    a.hist = (s->order == 2) ? s->d_hist : nullptr;
    a.o2_have = s->o2_have ? 1 : 0;
    return a;
}

// capture GRAPH_STEPS (node gather, cell step) pairs whose per-step data come from d_desc[k]
void drop_graphs(ep_sim* s) {
    for (cudaGraphExec_t& g : s->graph) if (g) { cudaGraphExecDestroy(g); g = nullptr; }
}

int build_graph(ep_sim* s, double dt) {
    if (s->graph_dt != dt || s->graph_model != s->model || s->graph_stream != s->stream) drop_graphs(s);
    cudaGraphExec_t& slot = s->graph[s->cur];
    if (slot) { cudaGraphExecDestroy(slot); slot = nullptr; }
    if (!s->d_desc) {
        EP_CUDA(s, cudaMalloc((void**)&s->d_desc, sizeof(epk::StepDesc) * GRAPH_STEPS));
        s->dev_bytes += (int64_t)sizeof(epk::StepDesc) * GRAPH_STEPS;
        EP_CUDA(s, cudaHostAlloc((void**)&s->h_desc, sizeof(epk::StepDesc) * GRAPH_STEPS * DESC_RING, cudaHostAllocDefault));
        for (int r = 0; r < DESC_RING; ++r) EP_CUDA(s, cudaEventCreateWithFlags(&s->desc_ev[r], cudaEventDisableTiming));
    }
    cudaGraph_t g = nullptr;
    EP_CUDA(s, cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
    int cur = s->cur;
    for (int k = 0; k < GRAPH_STEPS; ++k) {
        epk::StepArgs a = step_args(s, cur, dt);
        a.desc = s->d_desc + k;
        epk::launch_node_gather(s->dm, a.vm_cur, s->d_vn, s->stream, s->pdl);
        epk::launch_cell_step(s->dm, s->model, a, s->stream, s->pdl);
        cur ^= 1;
    }
    EP_CUDA(s, cudaStreamEndCapture(s->stream, &g));
    cudaError_t e = cudaGraphInstantiate(&slot, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { slot = nullptr; EP_CUDA(s, e); }
    s->graph_dt = dt; s->graph_model = s->model; s->graph_stream = s->stream;
    return EP_OK;
}

// every entry point that touches the device goes through this: the handle's device becomes the current one
int use_device(ep_sim* s) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != s->device) {
        if (cudaSetDevice(s->device) != cudaSuccess) {
            cudaGetLastError();
            return fail(EP_ERR_CUDA, "cannot make the handle's device current");
        }
    }
    return EP_OK;
}

int check_sim(ep_sim* s) {
    int rc = use_device(s);
    if (rc) return rc;
    if (s->sticky != EP_OK) return fail(s->sticky, "sim is in a sticky error state: " + g_err);
    return EP_OK;
}

// device (permuted) array -> host array in the caller's order
int read_back(ep_sim* s, const double* d_src, double* out) {
    epk::launch_gather_f64(s->nc, d_src, s->d_inv, s->d_tmp, s->stream);
    s->launches++;
    EP_CUDA(s, cudaMemcpyAsync(out, s->d_tmp, sizeof(double) * s->nc, cudaMemcpyDeviceToHost, s->stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    return EP_OK;
}

// Bidomain: v_ext for the potential in d_vm[cur] (second equation of (6)), then the coupling term of the next
// step.  Both sides are multiplied by the cell volumes (flux form: the operator then has the constants as left AND right
// null vectors, which is what makes GMRES safe on this singular, compatible system); gauge: zero volume-weighted mean.
int bidomain_solve(ep_sim* s) {
    if (!s->gm.V) {
        if (epk::gmres_alloc(s->gm, s->nc, s->bd_restart) != 0) {
            epk::gmres_free(s->gm);
            cudaGetLastError();
            return fail(EP_ERR_NOMEM, "cannot allocate the Krylov basis of the bidomain solver");
        }
        s->dev_bytes += s->gm.bytes;
    }
    const double* v = s->d_vm[s->cur];
    epk::launch_node_gather(s->dm, v, s->d_vn, s->stream);
    epk::launch_diffusion_only(s->dm, v, s->d_vn, s->d_b, s->stream, nullptr, s->d_vol, -1.0);   // b = -V A_i v
    // sum_c b_c = 0 analytically (conservation); what round-off leaves is removed so that the system stays compatible
    epk::launch_remove_mean(s->gm, s->d_b, s->stream);
    s->launches += 5;
    epk::GmresOp op;
    op.launches = 2;
    op.f = [s](const double* x, double* out, cudaStream_t st) {
        epk::launch_node_gather(s->dm, x, s->d_vn, st);
        epk::launch_diffusion_only(s->dm, x, s->d_vn, out, st, s->d_ccoef_ie, s->d_vol, 1.0);      // V A_ie x
    };
    // first estimate: the paper uses v_ext^n; with two previous solutions at hand their linear extrapolation
    // 2 v_ext^n - v_ext^{n-1} starts one order in dt closer (the gauge is preserved: both have zero weighted mean)
    epk::launch_extrapolate(s->nc, s->d_vext, s->d_vext_prev, s->vext_hist >= 2 ? 1 : 0, s->stream);
    s->launches++;
    double rel = 0.0;
    // reading E3: besides the relative criterion the solve stops at a residual density of rel_tol * 0.1 mV/ms (1e-11 mV/ms at
    // the default), the level at which the coupling term is exact for the purposes of the Vm update; a right-hand side that
    // is pure round-off (uniform potential) is met by the first estimate at once
    const double abs_tol = s->bd_tol * 0.1 * s->vol_norm2;
    const int it = epk::gmres_solve(s->gm, op, s->d_b, s->d_vext, s->bd_tol, abs_tol, s->bd_max_cycles, s->bd_check, s->stream,
                                    &rel, &s->launches);
    if (it < 0) {
        s->sticky = EP_ERR_CUDA;
        return fail(EP_ERR_CUDA, std::string("bidomain solver: ") + cudaGetErrorString(cudaGetLastError()));
    }
    s->bd_iters_last = it; s->bd_iters_total += it; s->bd_solves += 1; s->bd_res_last = rel;
    if (!(rel <= s->bd_tol)) {
        s->sticky = EP_ERR_NUMERIC;
        char msg[160];
        std::snprintf(msg, sizeof msg, "bidomain solver did not converge: relative residual %.3e after %d iterations", rel, it);
        return fail(EP_ERR_NUMERIC, msg);
    }
    epk::launch_remove_weighted_mean(s->gm, s->d_vext, s->d_vol, s->vol_total, s->stream);
    epk::launch_node_gather(s->dm, s->d_vext, s->d_vn, s->stream);
    epk::launch_diffusion_only(s->dm, s->d_vext, s->d_vn, s->d_src, s->stream);                  // A_i v_ext/(chi Cm), mV/ms
    s->launches += 5;
    s->vext_valid = true;
    if (s->vext_hist < 2) s->vext_hist++;
    return EP_OK;
}

}  // namespace

namespace ep {
// for the other translation units of the library (ep_noalloc.cu): record the message ep_last_error() returns
int set_error(int code, const char* msg) { return fail(code, msg ? msg : ""); }
}  // namespace ep

extern "C" {

const char* ep_last_error(void) { return g_err.c_str(); }

int ep_model_n_states(int model) { return epk::model_n_states(model); }

int ep_host_stencil(int64_t n_nodes, const double* xyz, int64_t n_tets, const int32_t* tets, const double* fibre,
                    const double* sigma_scale, double sigma_l, double sigma_t, double chi, double Cm, int32_t* node,
                    double* a, int32_t* nbr, double* b, int64_t* node_ptr, int32_t* node_cell, double* w,
                    int32_t* perm) {
    try {
        ep::Stencil st;
        std::string err;
        int rc = ep::build_stencil(n_nodes, xyz, n_tets, tets, fibre, sigma_scale, sigma_l, sigma_t, chi, Cm, st, err);
        if (rc) return fail(rc, err);
        if (node) std::memcpy(node, st.node.data(), sizeof(int32_t) * st.node.size());
        if (a) std::memcpy(a, st.a.data(), sizeof(double) * st.a.size());
        if (nbr) std::memcpy(nbr, st.nbr.data(), sizeof(int32_t) * st.nbr.size());
        if (b) std::memcpy(b, st.b.data(), sizeof(double) * st.b.size());
        if (node_ptr) std::memcpy(node_ptr, st.node_ptr.data(), sizeof(int64_t) * st.node_ptr.size());
        if (node_cell) std::memcpy(node_cell, st.node_cell.data(), sizeof(int32_t) * st.node_cell.size());
        if (w) std::memcpy(w, st.w.data(), sizeof(double) * st.w.size());
        if (perm) {
            ep::Packed pk;
            rc = ep::pack(st, xyz, pk, err);
            if (rc) return fail(rc, err);
            std::memcpy(perm, pk.perm_c.data(), sizeof(int32_t) * pk.perm_c.size());
        }
        return EP_OK;
    } catch (const std::bad_alloc&) {
        return fail(EP_ERR_NOMEM, "host allocation failed");
    } catch (...) {
        return fail(EP_ERR_ARG, "unexpected exception in preprocessor");
    }
}

// dim = 3: tetrahedra (cells [n*4]); dim = 2: triangles (cells [n*3])
// ext_l, ext_t > 0: bidomain; (sigma_l, sigma_t) are then the intracellular conductivities
static int mesh_create_impl(ep_sim** out, int dim, int64_t n_nodes, const double* xyz, int64_t n_tets, const int32_t* tets,
                            const double* fibre, const double* sigma_scale, double sigma_l, double sigma_t, double chi,
                            double Cm, double ext_l = 0.0, double ext_t = 0.0, int64_t n_owned = -1) {
    if (!out) return fail(EP_ERR_ARG, "out is NULL");
    *out = nullptr;
    ep_sim* s = nullptr;
    try {
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
            cudaGetLastError();
            return fail(EP_ERR_CUDA, "no CUDA device: libep has no CPU fallback");
        }
        ep::Stencil st;
        ep::Packed pk;
        std::string err;
        int rc = dim == 3 ? ep::build_stencil(n_nodes, xyz, n_tets, tets, fibre, sigma_scale, sigma_l, sigma_t, chi, Cm, st, err)
                          : ep::build_stencil_tri(n_nodes, xyz, n_tets, tets, fibre, sigma_scale, sigma_l, sigma_t, chi, Cm, st, err);
        if (rc) return fail(rc, err);
        rc = ep::pack(st, xyz, pk, err, n_owned);
        if (rc) return fail(rc, err);
        s = new ep_sim();
        s->dim = dim;
        s->n_owned = (n_owned >= 0 && n_owned < n_tets) ? n_owned : n_tets;
        cudaGetDevice(&s->device);
        s->pdl = (std::getenv("EP_NO_PDL") == nullptr);
        s->nc = pk.nc; s->nn = pk.nn; s->nc_pad = pk.nc_pad; s->chi = chi; s->Cm = Cm;
        s->star_entries = pk.star_entries;
        s->vol_total = pk.vol_total;
        for (double vv : pk.vol) s->vol_norm2 += vv * vv;
        s->vol_norm2 = std::sqrt(s->vol_norm2);
        s->perm_c = pk.perm_c; s->inv_c = pk.inv_c;
        s->smask_host.assign(s->nc_pad, 0);
        auto bail = [&](int code) { free_all(s); delete s; return code; };
        if (cudaStreamCreateWithFlags(&s->own_stream, cudaStreamNonBlocking) != cudaSuccess)
            return bail(fail(EP_ERR_CUDA, "cudaStreamCreate failed"));
        s->stream = s->own_stream;
        if ((rc = upload(s, &s->d_cidx, pk.cidx)) || (rc = upload(s, &s->d_ccoef, pk.ccoef)) ||
            (rc = upload(s, &s->d_slice_ptr, pk.slice_ptr)) || (rc = upload(s, &s->d_nidx, pk.nidx)) ||
            (rc = upload(s, &s->d_nw, pk.nw)) || (rc = upload(s, &s->d_perm, pk.perm_c)) ||
            (rc = upload(s, &s->d_inv, pk.inv_c)) || (rc = upload(s, &s->d_vol, pk.vol)))
            return bail(rc);
        if ((rc = dev_alloc(s, &s->d_vm[0], s->nc_pad)) || (rc = dev_alloc(s, &s->d_vm[1], s->nc_pad)) ||
            (rc = dev_alloc(s, &s->d_vn, s->nn)) || (rc = dev_alloc(s, &s->d_tact, s->nc_pad)) ||
            (rc = dev_alloc(s, &s->d_tmp, s->nc_pad)) || (rc = dev_alloc(s, &s->d_tmp2, s->nc_pad)) ||
            (rc = dev_alloc(s, &s->d_red, 1024 + 8)) || (rc = dev_alloc(s, &s->d_ctype, s->nc_pad)) ||
            (rc = dev_alloc(s, &s->d_smask, s->nc_pad)))
            return bail(rc);
        cudaMemset(s->d_vm[0], 0, sizeof(double) * s->nc_pad);
        cudaMemset(s->d_vm[1], 0, sizeof(double) * s->nc_pad);
        cudaMemset(s->d_ctype, 0, s->nc_pad);
        cudaMemset(s->d_smask, 0, s->nc_pad);
        s->tmask_host.assign(s->nc_pad, 0);
        if ((rc = dev_alloc(s, &s->d_tmask, s->nc_pad)) || (rc = dev_alloc(s, &s->d_trig_fire, epk::MAX_TRIGGERS)) ||
            (rc = dev_alloc(s, &s->d_trig_par, epk::MAX_TRIGGERS)))
            return bail(rc);
        cudaMemset(s->d_tmask, 0, s->nc_pad);
        cudaMemset(s->d_trig_fire, 0xff, sizeof(long long) * epk::MAX_TRIGGERS);
        cudaMemset(s->d_trig_par, 0, sizeof(epk::TrigPar) * epk::MAX_TRIGGERS);
        s->dm.nc = s->nc; s->dm.nn = s->nn; s->dm.nc_pad = s->nc_pad; s->dm.n_slices = pk.n_slices;
        s->dm.nc_active = s->n_owned;
        s->dm.cidx = s->d_cidx; s->dm.ccoef = s->d_ccoef; s->dm.slice_ptr = s->d_slice_ptr;
        s->dm.nidx = s->d_nidx; s->dm.nw = s->d_nw;
        if (ext_l > 0.0 || ext_t > 0.0) {
            if (!(ext_l > 0.0) || !(ext_t > 0.0)) return bail(fail(EP_ERR_ARG, "extracellular conductivities must be positive"));
            ep::Stencil st2;
            ep::Packed pk2;
            rc = ep::build_stencil(n_nodes, xyz, n_tets, tets, fibre, sigma_scale, sigma_l + ext_l, sigma_t + ext_t, chi, Cm, st2, err);
            if (rc) return bail(fail(rc, err));
            rc = ep::pack(st2, xyz, pk2, err, n_owned);
            if (rc) return bail(fail(rc, err));
            if (pk2.cidx != pk.cidx) return bail(fail(EP_ERR_MESH, "internal: index tables of the two operators differ"));
            if ((rc = upload(s, &s->d_ccoef_ie, pk2.ccoef)) || (rc = dev_alloc(s, &s->d_vext, s->nc_pad)) ||
                (rc = dev_alloc(s, &s->d_src, s->nc_pad)) || (rc = dev_alloc(s, &s->d_b, s->nc_pad)) ||
                (rc = dev_alloc(s, &s->d_vext_prev, s->nc_pad)))
                return bail(rc);
            cudaMemset(s->d_vext, 0, sizeof(double) * s->nc_pad);
            cudaMemset(s->d_src, 0, sizeof(double) * s->nc_pad);
            cudaMemset(s->d_b, 0, sizeof(double) * s->nc_pad);
            s->bidomain = true;
        }
        if (cudaDeviceSynchronize() != cudaSuccess) return bail(fail(EP_ERR_CUDA, "upload failed"));
        *out = s;
        return EP_OK;
    } catch (const std::bad_alloc&) {
        if (s) { free_all(s); delete s; }
        return fail(EP_ERR_NOMEM, "host allocation failed");
    } catch (...) {
        if (s) { free_all(s); delete s; }
        return fail(EP_ERR_ARG, "unexpected exception");
    }
}

int ep_host_stencil_tri(int64_t n_nodes, const double* xyz, int64_t n_tris, const int32_t* tris, const double* fibre,
                        const double* sigma_scale, double sigma_l, double sigma_t, double chi, double Cm, int32_t* node,
                        double* a, int32_t* nbr, double* b, int64_t* node_ptr, int32_t* node_cell, double* w,
                        int32_t* perm) {
    try {
        ep::Stencil st;
        std::string err;
        int rc = ep::build_stencil_tri(n_nodes, xyz, n_tris, tris, fibre, sigma_scale, sigma_l, sigma_t, chi, Cm, st, err);
        if (rc) return fail(rc, err);
        if (node) std::memcpy(node, st.node.data(), sizeof(int32_t) * st.node.size());
        if (a) std::memcpy(a, st.a.data(), sizeof(double) * st.a.size());
        if (nbr) std::memcpy(nbr, st.nbr.data(), sizeof(int32_t) * st.nbr.size());
        if (b) std::memcpy(b, st.b.data(), sizeof(double) * st.b.size());
        if (node_ptr) std::memcpy(node_ptr, st.node_ptr.data(), sizeof(int64_t) * st.node_ptr.size());
        if (node_cell) std::memcpy(node_cell, st.node_cell.data(), sizeof(int32_t) * st.node_cell.size());
        if (w) std::memcpy(w, st.w.data(), sizeof(double) * st.w.size());
        if (perm) {
            ep::Packed pk;
            rc = ep::pack(st, xyz, pk, err);
            if (rc) return fail(rc, err);
            std::memcpy(perm, pk.perm_c.data(), sizeof(int32_t) * pk.perm_c.size());
        }
        return EP_OK;
    } catch (const std::bad_alloc&) {
        return fail(EP_ERR_NOMEM, "host allocation failed");
    } catch (...) {
        return fail(EP_ERR_ARG, "unexpected exception in preprocessor");
    }
}

int ep_mesh_create(ep_sim** out, int64_t n_nodes, const double* xyz, int64_t n_tets, const int32_t* tets,
                   const double* fibre, const double* sigma_scale, double sigma_l, double sigma_t, double chi,
                   double Cm) {
    return mesh_create_impl(out, 3, n_nodes, xyz, n_tets, tets, fibre, sigma_scale, sigma_l, sigma_t, chi, Cm);
}

int ep_mesh_create_tri(ep_sim** out, int64_t n_nodes, const double* xyz, int64_t n_tris, const int32_t* tris,
                       const double* fibre, const double* sigma_scale, double sigma_l, double sigma_t, double chi,
                       double Cm) {
    return mesh_create_impl(out, 2, n_nodes, xyz, n_tris, tris, fibre, sigma_scale, sigma_l, sigma_t, chi, Cm);
}

int ep_mesh_create_bidomain(ep_sim** out, int64_t n_nodes, const double* xyz, int64_t n_tets, const int32_t* tets,
                            const double* fibre, const double* sigma_scale, double sigma_int_l, double sigma_int_t,
                            double sigma_ext_l, double sigma_ext_t, double chi, double Cm) {
    if (!(sigma_ext_l > 0.0) || !(sigma_ext_t > 0.0)) return fail(EP_ERR_ARG, "extracellular conductivities must be positive");
    return mesh_create_impl(out, 3, n_nodes, xyz, n_tets, tets, fibre, sigma_scale, sigma_int_l, sigma_int_t, chi, Cm,
                            sigma_ext_l, sigma_ext_t);
}

int ep_shard_plan(int64_t n_nodes, const double* xyz, int64_t n_tets, const int32_t* tets, int part, int n_parts,
                  int64_t* counts, int64_t* local_cells, int64_t* send_ptr, int64_t* send_global, int64_t* recv_ptr,
                  int64_t* recv_global) {
    if (!counts) return fail(EP_ERR_ARG, "counts is NULL");
    try {
        ep::ShardPlan pl;
        std::string err;
        int rc = ep::shard_plan(n_nodes, xyz, n_tets, tets, part, n_parts, pl, err);
        if (rc) return fail(rc, err);
        counts[0] = pl.n_owned; counts[1] = (int64_t)pl.local_cells.size();
        counts[2] = (int64_t)pl.send_cells.size(); counts[3] = (int64_t)pl.recv_cells.size();
        if (local_cells) std::memcpy(local_cells, pl.local_cells.data(), sizeof(int64_t) * pl.local_cells.size());
        if (send_ptr) std::memcpy(send_ptr, pl.send_ptr.data(), sizeof(int64_t) * pl.send_ptr.size());
        if (recv_ptr) std::memcpy(recv_ptr, pl.recv_ptr.data(), sizeof(int64_t) * pl.recv_ptr.size());
        if (send_global) for (size_t k = 0; k < pl.send_cells.size(); ++k) send_global[k] = pl.local_cells[pl.send_cells[k]];
        if (recv_global) for (size_t k = 0; k < pl.recv_cells.size(); ++k) recv_global[k] = pl.local_cells[pl.recv_cells[k]];
        return EP_OK;
    } catch (const std::bad_alloc&) {
        return fail(EP_ERR_NOMEM, "host allocation failed");
    } catch (...) {
        return fail(EP_ERR_ARG, "unexpected exception in the partitioner");
    }
}

int ep_shard_create(ep_sim** out, int64_t n_nodes, const double* xyz, int64_t n_tets, const int32_t* tets,
                    const double* fibre, const double* sigma_scale, double sigma_l, double sigma_t, double chi, double Cm,
                    int part, int n_parts) {
    if (!out) return fail(EP_ERR_ARG, "out is NULL");
    *out = nullptr;
    try {
        ep::ShardPlan pl;
        std::string err;
        int rc = ep::shard_plan(n_nodes, xyz, n_tets, tets, part, n_parts, pl, err);
        if (rc) return fail(rc, err);
        const int64_t nl = (int64_t)pl.local_cells.size(), nln = (int64_t)pl.local_nodes.size();
        std::vector<double> lxyz(3 * nln), lfib, lscale;
        for (int64_t k = 0; k < nln; ++k)
            for (int d = 0; d < 3; ++d) lxyz[3 * k + d] = xyz[3 * pl.local_nodes[k] + d];
        if (fibre) {
            lfib.resize(3 * nl);
            for (int64_t k = 0; k < nl; ++k)
                for (int d = 0; d < 3; ++d) lfib[3 * k + d] = fibre[3 * pl.local_cells[k] + d];
        }
        if (sigma_scale) {
            lscale.resize(nl);
            for (int64_t k = 0; k < nl; ++k) lscale[k] = sigma_scale[pl.local_cells[k]];
        }
        ep_sim* s = nullptr;
        rc = mesh_create_impl(&s, 3, nln, lxyz.data(), nl, pl.local_tets.data(), fibre ? lfib.data() : nullptr,
                              sigma_scale ? lscale.data() : nullptr, sigma_l, sigma_t, chi, Cm, 0.0, 0.0, pl.n_owned);
        if (rc) return rc;
        s->n_parts = n_parts; s->part = part;
        s->shard_global = pl.local_cells;
        s->send_ptr = pl.send_ptr; s->recv_ptr = pl.recv_ptr;
        std::vector<int32_t> si(pl.send_cells.size()), ri(pl.recv_cells.size());
        for (size_t k = 0; k < si.size(); ++k) si[k] = s->inv_c[pl.send_cells[k]];
        for (size_t k = 0; k < ri.size(); ++k) ri[k] = s->inv_c[pl.recv_cells[k]];
        if ((rc = upload(s, &s->d_send_idx, si)) || (rc = upload(s, &s->d_recv_idx, ri)) ||
            (rc = dev_alloc(s, &s->d_send, (int64_t)si.size())) || (rc = dev_alloc(s, &s->d_recv, (int64_t)ri.size()))) {
            free_all(s); delete s;
            return rc;
        }
        *out = s;
        return EP_OK;
    } catch (const std::bad_alloc&) {
        return fail(EP_ERR_NOMEM, "host allocation failed");
    } catch (...) {
        return fail(EP_ERR_ARG, "unexpected exception");
    }
}

int ep_shard_info(ep_sim* s, int64_t* n_owned, int64_t* n_local, int64_t* global_ids, int64_t* send_ptr, int64_t* recv_ptr) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (s->shard_global.empty()) return fail(EP_ERR_STATE, "not a shard (ep_shard_create)");
    if (n_owned) *n_owned = s->n_owned;
    if (n_local) *n_local = s->nc;
    if (global_ids) std::memcpy(global_ids, s->shard_global.data(), sizeof(int64_t) * s->shard_global.size());
    if (send_ptr) std::memcpy(send_ptr, s->send_ptr.data(), sizeof(int64_t) * s->send_ptr.size());
    if (recv_ptr) std::memcpy(recv_ptr, s->recv_ptr.data(), sizeof(int64_t) * s->recv_ptr.size());
    return EP_OK;
}

int ep_shard_buffers(ep_sim* s, void** send_dptr, void** recv_dptr) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (s->shard_global.empty()) return fail(EP_ERR_STATE, "not a shard (ep_shard_create)");
    if (send_dptr) *send_dptr = s->d_send;
    if (recv_dptr) *recv_dptr = s->d_recv;
    return EP_OK;
}

int ep_halo_pack(ep_sim* s) {
    int rc = check_sim(s);
    if (rc) return rc;
    if (s->shard_global.empty()) return fail(EP_ERR_STATE, "not a shard (ep_shard_create)");
    const int64_t n = s->send_ptr.back();
    if (n > 0) { epk::launch_gather_f64(n, s->d_vm[s->cur], s->d_send_idx, s->d_send, s->stream); s->launches++; }
    EP_CUDA(s, cudaGetLastError());
    return EP_OK;
}

int ep_halo_unpack(ep_sim* s) {
    int rc = check_sim(s);
    if (rc) return rc;
    if (s->shard_global.empty()) return fail(EP_ERR_STATE, "not a shard (ep_shard_create)");
    const int64_t n = s->recv_ptr.back();
    if (n > 0) { epk::launch_scatter_f64(n, s->d_recv, s->d_recv_idx, s->d_vm[s->cur], s->stream); s->launches++; }
    EP_CUDA(s, cudaGetLastError());
    return EP_OK;
}

int ep_halo_exchange_local(ep_sim** sims, int n) {
    if (!sims || n < 1) return fail(EP_ERR_ARG, "bad shard list");
    for (int p = 0; p < n; ++p) {
        if (!sims[p] || sims[p]->shard_global.empty() || sims[p]->n_parts != n || sims[p]->part != p)
            return fail(EP_ERR_ARG, "sims[p] must be part p of an n-part sharding");
    }
    int rc;
    for (int p = 0; p < n; ++p) if ((rc = ep_halo_pack(sims[p]))) return rc;
    for (int p = 0; p < n; ++p) EP_CUDA(sims[p], cudaStreamSynchronize(sims[p]->stream));
    for (int p = 0; p < n; ++p)          // p receives from q what q sends to p: same cells, same order
        for (int q = 0; q < n; ++q) {
            const int64_t cnt = sims[p]->recv_ptr[q + 1] - sims[p]->recv_ptr[q];
            if (cnt != sims[q]->send_ptr[p + 1] - sims[q]->send_ptr[p]) return fail(EP_ERR_STATE, "exchange lists do not match");
            if (cnt == 0) continue;
            EP_CUDA(sims[p], cudaMemcpyAsync(sims[p]->d_recv + sims[p]->recv_ptr[q], sims[q]->d_send + sims[q]->send_ptr[p],
                                             sizeof(double) * cnt, cudaMemcpyDeviceToDevice, sims[p]->stream));
        }
    for (int p = 0; p < n; ++p) if ((rc = ep_halo_unpack(sims[p]))) return rc;
    return EP_OK;
}

void ep_destroy(ep_sim* s) {
    if (!s) return;
    cudaStreamSynchronize(s->stream);
    free_all(s);
    delete s;
}

int ep_set_stream(ep_sim* s, void* cuda_stream) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    cudaStreamSynchronize(s->stream);
    s->stream = cuda_stream ? (cudaStream_t)cuda_stream : s->own_stream;
    return EP_OK;
}

int ep_state_init(ep_sim* s, int model, const uint8_t* cell_type, const double* y0) {
    int rc = use_device(s);
    if (rc) return rc;
    if (s->sticky == EP_ERR_CUDA) return fail(EP_ERR_CUDA, "sim is in a sticky CUDA error state");
    const int S = epk::model_n_states(model);
    if (S < 0) return fail(EP_ERR_ARG, "unknown cell model");
    const int n_types = (model == EP_MODEL_TP06) ? 3 : 1;   // Courtemanche and Stewart have one cell type
    if (y0)
        for (int k = 0; k < n_types * S; ++k)
            if (!std::isfinite(y0[k])) return fail(EP_ERR_ARG, "non-finite initial state");
    // ep_step is asynchronous on a non-blocking stream: nothing below may overtake a step kernel still in flight
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    try {
        std::vector<uint8_t> ct(s->nc_pad, 0);
        if (cell_type) {
            for (int64_t i = 0; i < s->nc; ++i) {
                const uint8_t t = cell_type[s->perm_c[i]];
                if (t >= n_types) return fail(EP_ERR_ARG, "cell_type out of range for this model");
                ct[i] = t;
            }
        }
        EP_CUDA(s, cudaMemcpyAsync(s->d_ctype, ct.data(), s->nc_pad, cudaMemcpyHostToDevice, s->stream));
        EP_CUDA(s, cudaStreamSynchronize(s->stream));   // ct goes out of scope
    } catch (const std::bad_alloc&) {
        return fail(EP_ERR_NOMEM, "host allocation failed");
    }
    if (s->S != S) {
        if (s->d_y) { cudaFree(s->d_y); s->dev_bytes -= (int64_t)sizeof(double) * s->S * s->nc_pad; s->d_y = nullptr; s->S = 0; }
        rc = dev_alloc(s, &s->d_y, (int64_t)S * s->nc_pad);
        if (rc) return rc;
        // row 0 of the state array is never used (Vm lives in vm[2]): define it so that whole-array checks see numbers
        EP_CUDA(s, cudaMemsetAsync(s->d_y, 0, sizeof(double) * (size_t)S * s->nc_pad, s->stream));
    }
    s->model = model; s->S = S; s->step = 0; s->dt = 0.0; s->cur = 0;
    s->o2_have = false;
    if (s->order == 2 && model != EP_MODEL_TP06) s->order = 1;   // the second-order scheme exists for TP06 only
    if (s->bidomain) {
        s->vext_valid = false;
        s->vext_hist = 0;
        EP_CUDA(s, cudaMemsetAsync(s->d_vext, 0, sizeof(double) * s->nc_pad, s->stream));
        EP_CUDA(s, cudaMemsetAsync(s->d_src, 0, sizeof(double) * s->nc_pad, s->stream));
    }
    if (s->sticky == EP_ERR_NUMERIC) s->sticky = EP_OK;   // a fresh state clears a numerical failure, not a CUDA one
    s->trig_dirty = true;
    double* d_y0 = nullptr;
    cudaError_t e = cudaSuccess;
    if (y0) {
        e = cudaMalloc((void**)&d_y0, sizeof(double) * n_types * S);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(d_y0, y0, sizeof(double) * n_types * S, cudaMemcpyHostToDevice, s->stream);
    }
    if (e == cudaSuccess)   // triggers back to "not fired"
        e = cudaMemsetAsync(s->d_trig_fire, 0xff, sizeof(long long) * epk::MAX_TRIGGERS, s->stream);
    if (e == cudaSuccess) {
        epk::launch_state_fill(model, s->nc, s->nc_pad, s->d_ctype, d_y0, s->d_y, s->d_vm[0], s->d_tact, s->stream);
        s->launches++;
        e = cudaMemcpyAsync(s->d_vm[1], s->d_vm[0], sizeof(double) * s->nc_pad, cudaMemcpyDeviceToDevice, s->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    if (d_y0) cudaFree(d_y0);
    EP_CUDA(s, e);
    return EP_OK;
}

int ep_stimulus_set(ep_sim* s, int slot, int64_t n_cells, const int64_t* cell_ids, double amp, double t0, double dur) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (slot < 0 || slot >= EP_MAX_STIM_SLOTS) return fail(EP_ERR_ARG, "stimulus slot out of range");
    if (n_cells < 0 || (n_cells > 0 && !cell_ids)) return fail(EP_ERR_ARG, "bad stimulus cell list");
    if (!std::isfinite(amp) || !std::isfinite(t0) || !std::isfinite(dur) || dur < 0.0)
        return fail(EP_ERR_ARG, "bad stimulus amplitude or window");
    for (int64_t k = 0; k < n_cells; ++k)
        if (cell_ids[k] < 0 || cell_ids[k] >= s->nc) return fail(EP_ERR_ARG, "stimulus cell id out of range");
    const uint8_t bit = (uint8_t)(1u << slot);
    for (int64_t i = 0; i < s->nc; ++i) s->smask_host[i] &= (uint8_t)~bit;
    for (int64_t k = 0; k < n_cells; ++k) s->smask_host[s->inv_c[cell_ids[k]]] |= bit;
    s->stim[slot].set = n_cells > 0;
    s->stim[slot].amp = amp; s->stim[slot].t0 = t0; s->stim[slot].dur = dur; s->stim[slot].n_cells = n_cells;
    s->trig_dirty = true;   // a trigger may drive this slot: its amplitude / duration are cached on the device
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    EP_CUDA(s, cudaMemcpy(s->d_smask, s->smask_host.data(), s->nc_pad, cudaMemcpyHostToDevice));
    return EP_OK;
}

int ep_step(ep_sim* s, int64_t n_steps, double dt) {
    int rc = check_sim(s);
    if (rc) return rc;
    if (s->model < 0) return fail(EP_ERR_STATE, "ep_step before ep_state_init");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(EP_ERR_STATE, "dt must be positive");
    if (n_steps < 0) return fail(EP_ERR_ARG, "n_steps must be non-negative");
    if (s->step > 0 && dt != s->dt) return fail(EP_ERR_STATE, "dt may not change after the first step");
    s->dt = dt;
    int64_t n_on[EP_MAX_STIM_SLOTS], n_off[EP_MAX_STIM_SLOTS];
    for (int k = 0; k < EP_MAX_STIM_SLOTS; ++k) {
        n_on[k] = n_off[k] = 0;
        if (!s->stim[k].set) continue;
        n_on[k] = step_index(s->stim[k].t0, dt);
        n_off[k] = step_index(s->stim[k].t0 + s->stim[k].dur, dt);
    }
    if (s->trig_dirty) {   // trigger parameters in steps of this dt; a changed trigger set invalidates the captured graph
        epk::TrigPar par[epk::MAX_TRIGGERS];
        for (int t = 0; t < epk::MAX_TRIGGERS; ++t) {
            const ep_sim::Trig& g = s->trig[t];
            const bool drives = g.armed && g.slot >= 0;   // slot -1: monitor only (cross-handle coupling, ep_couple)
            par[t].armed = g.armed ? 1 : 0;
            par[t].slot = g.slot;
            par[t].nd = (int32_t)step_index(g.delay, dt);
            par[t].ndur = drives ? (int32_t)step_index(s->stim[g.slot].dur, dt) : 0;
            par[t].amp_cm = drives ? s->stim[g.slot].amp / s->Cm : 0.0;
        }
        EP_CUDA(s, cudaStreamSynchronize(s->stream));
        EP_CUDA(s, cudaMemcpy(s->d_trig_par, par, sizeof(par), cudaMemcpyHostToDevice));
        drop_graphs(s);
        s->trig_dirty = false;
    }
    int64_t left = n_steps;
    if (s->bidomain) {
        // v^{n+1} explicit from v, v_ext, I_ion, I_s at t^n, then the elliptic solve for v_ext^{n+1}
        if (left > 0 && !s->vext_valid && (rc = bidomain_solve(s))) return rc;     // reading E2: v_ext^0 from v^0
        for (; left > 0; --left) {
            epk::StepArgs a = step_args(s, s->cur, dt);
            fill_desc(s, s->step, dt, n_on, n_off, a.inl);
            epk::launch_node_gather(s->dm, a.vm_cur, s->d_vn, s->stream);
            epk::launch_cell_step(s->dm, s->model, a, s->stream);
            s->launches += 2;
            s->cur ^= 1;
            s->step += 1;
            if (s->order == 2) s->o2_have = true;
            if ((rc = bidomain_solve(s))) return rc;
        }
        EP_CUDA(s, cudaGetLastError());
        return EP_OK;
    }
    while (left > 0) {
        if (!s->profiling && left >= GRAPH_STEPS && !(s->order == 2 && !s->o2_have)) {
            // replay path: one descriptor upload + one graph launch per GRAPH_STEPS time steps
            if (!s->graph[s->cur] || s->graph_dt != dt || s->graph_model != s->model || s->graph_stream != s->stream) {
                if ((rc = build_graph(s, dt))) return rc;
            }
            // pinned ring slot: wait (normally not at all) until the copy that last used it has run, refill, enqueue the
            // copy; stream order keeps the copy behind the previous replay and ahead of the next one
            const int r = s->desc_slot;
            s->desc_slot = (r + 1) % DESC_RING;
            if (s->desc_ev_used[r]) EP_CUDA(s, cudaEventSynchronize(s->desc_ev[r]));
            epk::StepDesc* h = s->h_desc + (size_t)r * GRAPH_STEPS;
            for (int k = 0; k < GRAPH_STEPS; ++k) fill_desc(s, s->step + k, dt, n_on, n_off, h[k]);
            EP_CUDA(s, cudaMemcpyAsync(s->d_desc, h, sizeof(epk::StepDesc) * GRAPH_STEPS, cudaMemcpyHostToDevice, s->stream));
            EP_CUDA(s, cudaEventRecord(s->desc_ev[r], s->stream));
            s->desc_ev_used[r] = true;
            EP_CUDA(s, cudaGraphLaunch(s->graph[s->cur], s->stream));
            s->launches += 2 * GRAPH_STEPS;
            s->step += GRAPH_STEPS;
            left -= GRAPH_STEPS;
            continue;
        }
        const int64_t n = s->step;
        epk::StepArgs a = step_args(s, s->cur, dt);
        fill_desc(s, n, dt, n_on, n_off, a.inl);
        if (s->profiling) {
            if (s->ev_used >= 3 * 4096 && (rc = profile_drain(s))) return rc;
            if ((rc = profile_event(s))) return rc;
            epk::launch_node_gather(s->dm, a.vm_cur, s->d_vn, s->stream);
            if ((rc = profile_event(s))) return rc;
            epk::launch_cell_step(s->dm, s->model, a, s->stream);
            if ((rc = profile_event(s))) return rc;
        } else {
            epk::launch_node_gather(s->dm, a.vm_cur, s->d_vn, s->stream, s->pdl);
            epk::launch_cell_step(s->dm, s->model, a, s->stream, s->pdl);
        }
        s->launches += 2;
        s->cur ^= 1;
        s->step = n + 1;
        --left;
        if (s->order == 2 && !s->o2_have) { s->o2_have = true; drop_graphs(s); }   // graphs bake the flag in
    }
    EP_CUDA(s, cudaGetLastError());
    return EP_OK;
}

int ep_synchronize(ep_sim* s) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    if (s->sticky != EP_OK) return fail(s->sticky, "sticky error");
    return EP_OK;
}

int ep_read_vm(ep_sim* s, double* out) { return ep_read_state(s, 0, out); }

int ep_read_state(ep_sim* s, int var, double* out) {
    if (!s || !out) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    if (var < 0 || var >= s->S) return fail(EP_ERR_ARG, "state variable index out of range");
    if (var == 0) return read_back(s, s->d_vm[s->cur], out);
    epk::launch_state_row_get(s->nc, s->d_y, s->S, var, s->d_inv, s->d_tmp, s->stream);
    s->launches++;
    EP_CUDA(s, cudaMemcpyAsync(out, s->d_tmp, sizeof(double) * s->nc, cudaMemcpyDeviceToHost, s->stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    return EP_OK;
}

int ep_write_state(ep_sim* s, int var, const double* in) {
    if (!s || !in) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    if (var < 0 || var >= s->S) return fail(EP_ERR_ARG, "state variable index out of range");
    EP_CUDA(s, cudaMemcpyAsync(s->d_tmp, in, sizeof(double) * s->nc, cudaMemcpyHostToDevice, s->stream));
    if (var == 0) epk::launch_gather_f64(s->nc, s->d_tmp, s->d_perm, s->d_vm[s->cur], s->stream);
    else epk::launch_state_row_put(s->nc, s->d_tmp, s->d_perm, s->S, var, s->d_y, s->stream);
    s->launches++;
    if (var == 0) { s->vext_valid = false; s->vext_hist = 0; }
    s->o2_have = false;      // a rewritten state has no history
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    return EP_OK;
}

int ep_activation_times(ep_sim* s, double* out) {
    if (!s || !out) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    int rc = use_device(s);
    if (rc) return rc;
    return read_back(s, s->d_tact, out);
}

int ep_write_activation_times(ep_sim* s, const double* in) {
    if (!s || !in) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    int rc = use_device(s);
    if (rc) return rc;
    EP_CUDA(s, cudaMemcpyAsync(s->d_tmp, in, sizeof(double) * s->nc, cudaMemcpyHostToDevice, s->stream));
    epk::launch_gather_f64(s->nc, s->d_tmp, s->d_perm, s->d_tact, s->stream);
    s->launches++;
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    return EP_OK;
}

int ep_set_step_count(ep_sim* s, int64_t step_count, double dt_ms) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    if (step_count < 0) return fail(EP_ERR_ARG, "step_count must be non-negative");
    if (step_count > 0 && (!(dt_ms > 0.0) || !std::isfinite(dt_ms))) return fail(EP_ERR_ARG, "dt must be positive");
    s->step = step_count;
    s->dt = step_count > 0 ? dt_ms : 0.0;
    return EP_OK;
}

int ep_trigger_restore(ep_sim* s, int trigger, double t_fire_ms) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (trigger < 0 || trigger >= epk::MAX_TRIGGERS) return fail(EP_ERR_ARG, "trigger index out of range");
    if (t_fire_ms >= 0.0 && !(s->dt > 0.0)) return fail(EP_ERR_STATE, "set the clock first (ep_set_step_count)");
    int rc = use_device(s);
    if (rc) return rc;
    const long long n1 = t_fire_ms < 0.0 ? -1 : (long long)std::llround(t_fire_ms / s->dt);
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    EP_CUDA(s, cudaMemcpy(s->d_trig_fire + trigger, &n1, sizeof(n1), cudaMemcpyHostToDevice));
    return EP_OK;
}

// Two-slot pipeline between the I/O stream (copies) and the sim's stream (permutation kernels): row k is copied while
// row k-1 is permuted; nothing synchronises with the host until the last row.
static int io_setup(ep_sim* s) {
    if (s->io_stream) return EP_OK;
    EP_CUDA(s, cudaStreamCreateWithFlags(&s->io_stream, cudaStreamNonBlocking));
    for (int k = 0; k < 2; ++k) {
        EP_CUDA(s, cudaEventCreateWithFlags(&s->io_copied[k], cudaEventDisableTiming));
        EP_CUDA(s, cudaEventCreateWithFlags(&s->io_consumed[k], cudaEventDisableTiming));
    }
    EP_CUDA(s, cudaEventCreateWithFlags(&s->io_fence, cudaEventDisableTiming));
    return EP_OK;
}

int ep_write_states(ep_sim* s, const double* in) {
    if (!s || !in) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    int rc = use_device(s);
    if (rc || (rc = io_setup(s))) return rc;
    double* stage[2] = {s->d_tmp, s->d_tmp2};
    EP_CUDA(s, cudaEventRecord(s->io_fence, s->stream));          // the staging buffers may still be in use by the sim's stream
    EP_CUDA(s, cudaStreamWaitEvent(s->io_stream, s->io_fence, 0));
    for (int k = 0; k < s->S; ++k) {
        const int b = k & 1;
        if (k >= 2) EP_CUDA(s, cudaStreamWaitEvent(s->io_stream, s->io_consumed[b], 0));
        EP_CUDA(s, cudaMemcpyAsync(stage[b], in + (size_t)k * s->nc, sizeof(double) * s->nc, cudaMemcpyHostToDevice, s->io_stream));
        EP_CUDA(s, cudaEventRecord(s->io_copied[b], s->io_stream));
        EP_CUDA(s, cudaStreamWaitEvent(s->stream, s->io_copied[b], 0));
        if (k == 0) epk::launch_gather_f64(s->nc, stage[b], s->d_perm, s->d_vm[s->cur], s->stream);
        else epk::launch_state_row_put(s->nc, stage[b], s->d_perm, s->S, k, s->d_y, s->stream);
        s->launches++;
        EP_CUDA(s, cudaEventRecord(s->io_consumed[b], s->stream));
    }
    s->vext_valid = false;
    s->vext_hist = 0;
    s->o2_have = false;
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    return EP_OK;
}

int ep_read_states(ep_sim* s, double* out) {
    if (!s || !out) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    int rc = use_device(s);
    if (rc || (rc = io_setup(s))) return rc;
    double* stage[2] = {s->d_tmp, s->d_tmp2};
    for (int k = 0; k < s->S; ++k) {
        const int b = k & 1;
        if (k >= 2) EP_CUDA(s, cudaStreamWaitEvent(s->stream, s->io_consumed[b], 0));
        if (k == 0) epk::launch_gather_f64(s->nc, s->d_vm[s->cur], s->d_inv, stage[b], s->stream);
        else epk::launch_state_row_get(s->nc, s->d_y, s->S, k, s->d_inv, stage[b], s->stream);
        s->launches++;
        EP_CUDA(s, cudaEventRecord(s->io_copied[b], s->stream));
        EP_CUDA(s, cudaStreamWaitEvent(s->io_stream, s->io_copied[b], 0));
        EP_CUDA(s, cudaMemcpyAsync(out + (size_t)k * s->nc, stage[b], sizeof(double) * s->nc, cudaMemcpyDeviceToHost, s->io_stream));
        EP_CUDA(s, cudaEventRecord(s->io_consumed[b], s->io_stream));
    }
    EP_CUDA(s, cudaStreamSynchronize(s->io_stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    return EP_OK;
}

int ep_apply_diffusion(ep_sim* s, const double* v, double* D) {
    if (!s || !v || !D) return fail(EP_ERR_ARG, "null argument");
    EP_CUDA(s, cudaMemcpyAsync(s->d_tmp, v, sizeof(double) * s->nc, cudaMemcpyHostToDevice, s->stream));
    epk::launch_gather_f64(s->nc, s->d_tmp, s->d_perm, s->d_tmp2, s->stream);
    epk::launch_node_gather(s->dm, s->d_tmp2, s->d_vn, s->stream);
    epk::launch_diffusion_only(s->dm, s->d_tmp2, s->d_vn, s->d_tmp, s->stream);
    epk::launch_gather_f64(s->nc, s->d_tmp, s->d_inv, s->d_tmp2, s->stream);
    s->launches += 4;
    EP_CUDA(s, cudaMemcpyAsync(D, s->d_tmp2, sizeof(double) * s->nc, cudaMemcpyDeviceToHost, s->stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    const double k = s->chi * s->Cm;   // the tables hold D/(chi Cm)
    for (int64_t c = 0; c < s->nc; ++c) D[c] *= k;
    return EP_OK;
}

int ep_stable_dt(ep_sim* s, double* dt_max) {
    if (!s || !dt_max) return fail(EP_ERR_ARG, "null argument");
    // power iteration on B = A/(chi Cm) [1/ms]: x <- Bx/|Bx|, rho ~ |Bx|; start from a fixed pseudo-random vector
    try {
        std::vector<double> x0(s->nc);
        uint64_t z = 0x9E3779B97F4A7C15ULL;
        for (int64_t i = 0; i < s->nc; ++i) {
            z ^= z << 13; z ^= z >> 7; z ^= z << 17;
            x0[i] = (double)(z >> 11) * (1.0 / 9007199254740992.0) - 0.5;
        }
        EP_CUDA(s, cudaMemcpyAsync(s->d_tmp, x0.data(), sizeof(double) * s->nc, cudaMemcpyHostToDevice, s->stream));
        EP_CUDA(s, cudaStreamSynchronize(s->stream));
    } catch (const std::bad_alloc&) {
        return fail(EP_ERR_NOMEM, "host allocation failed");
    }
    // |Bx_k| with |x_k| = 1 settles at rho; read it back every CHECK iterations and stop once it has stopped moving
    // (relative change below 1e-4 over CHECK iterations) or after MAX_ITERS.
    double rho = 0.0, rho_prev = 0.0;
    const int MAX_ITERS = 300, CHECK = 20;
    for (int it = 0; it < MAX_ITERS; ++it) {
        epk::launch_norm2(s->nc, s->d_tmp, s->d_red, s->d_red + 1024, s->stream);
        if (it > 0 && it % CHECK == 0) {
            double n2 = 0.0;
            EP_CUDA(s, cudaMemcpyAsync(&n2, s->d_red + 1024, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
            EP_CUDA(s, cudaStreamSynchronize(s->stream));
            rho = std::sqrt(n2);
            if (it > CHECK && std::fabs(rho - rho_prev) <= 1e-4 * rho) break;
            rho_prev = rho;
        }
        epk::launch_scale_by_inv_norm(s->nc, s->d_tmp, s->d_red + 1024, s->d_tmp2, s->stream);
        epk::launch_node_gather(s->dm, s->d_tmp2, s->d_vn, s->stream);
        epk::launch_diffusion_only(s->dm, s->d_tmp2, s->d_vn, s->d_tmp, s->stream);
        s->launches += 5;
    }
    epk::launch_norm2(s->nc, s->d_tmp, s->d_red, s->d_red + 1024, s->stream);
    s->launches += 2;
    double n2 = 0.0;
    EP_CUDA(s, cudaMemcpyAsync(&n2, s->d_red + 1024, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    rho = std::max(rho, std::sqrt(n2));
    if (!(rho > 0.0) || !std::isfinite(rho)) return fail(EP_ERR_NUMERIC, "power iteration failed");
    *dt_max = 2.0 / rho;
    return EP_OK;
}

int ep_trigger_set(ep_sim* s, int trigger, int64_t n_monitor, const int64_t* monitor_ids, int slot, double delay_ms) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (trigger < 0 || trigger >= epk::MAX_TRIGGERS) return fail(EP_ERR_ARG, "trigger index out of range");
    if (n_monitor < 0 || (n_monitor > 0 && !monitor_ids)) return fail(EP_ERR_ARG, "bad monitor cell list");
    if (n_monitor > 0 && (slot < -1 || slot >= EP_MAX_STIM_SLOTS)) return fail(EP_ERR_ARG, "stimulus slot out of range");
    if (!std::isfinite(delay_ms) || delay_ms < 0.0) return fail(EP_ERR_ARG, "delay must be finite and non-negative");
    for (int64_t k = 0; k < n_monitor; ++k)
        if (monitor_ids[k] < 0 || monitor_ids[k] >= s->nc) return fail(EP_ERR_ARG, "monitor cell id out of range");
    for (int t = 0; t < epk::MAX_TRIGGERS; ++t)
        if (n_monitor > 0 && slot >= 0 && t != trigger && s->trig[t].armed && s->trig[t].slot == slot)
            return fail(EP_ERR_ARG, "stimulus slot is already driven by another trigger");
    const uint8_t bit = (uint8_t)(1u << trigger);
    for (int64_t i = 0; i < s->nc; ++i) s->tmask_host[i] &= (uint8_t)~bit;
    for (int64_t k = 0; k < n_monitor; ++k) s->tmask_host[s->inv_c[monitor_ids[k]]] |= bit;
    s->trig[trigger].armed = n_monitor > 0;
    s->trig[trigger].slot = slot;
    s->trig[trigger].delay = delay_ms;
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    EP_CUDA(s, cudaMemcpy(s->d_tmask, s->tmask_host.data(), s->nc_pad, cudaMemcpyHostToDevice));
    const long long none = -1;
    EP_CUDA(s, cudaMemcpy(s->d_trig_fire + trigger, &none, sizeof(none), cudaMemcpyHostToDevice));
    s->trig_dirty = true;
    return EP_OK;
}

int ep_trigger_time(ep_sim* s, int trigger, double* t_fire_ms) {
    if (!s || !t_fire_ms) return fail(EP_ERR_ARG, "null argument");
    if (trigger < 0 || trigger >= epk::MAX_TRIGGERS) return fail(EP_ERR_ARG, "trigger index out of range");
    long long n1 = -1;
    EP_CUDA(s, cudaMemcpyAsync(&n1, s->d_trig_fire + trigger, sizeof(n1), cudaMemcpyDeviceToHost, s->stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    *t_fire_ms = n1 < 0 ? -1.0 : (double)n1 * s->dt;
    return EP_OK;
}

int ep_couple(ep_sim* src, int trigger, ep_sim* dst, int slot, double delay_ms, int* scheduled) {
    if (!src || !dst || !scheduled) return fail(EP_ERR_ARG, "null argument");
    if (slot < 0 || slot >= EP_MAX_STIM_SLOTS) return fail(EP_ERR_ARG, "stimulus slot out of range");
    if (!std::isfinite(delay_ms) || delay_ms < 0.0) return fail(EP_ERR_ARG, "delay must be finite and non-negative");
    if (!dst->stim[slot].set) return fail(EP_ERR_STATE, "destination slot has no cells: call ep_stimulus_set first");
    *scheduled = 0;
    double t_fire = -1.0;
    int rc = ep_trigger_time(src, trigger, &t_fire);
    if (rc) return rc;
    if (t_fire < 0.0) return EP_OK;
    const double t_on = t_fire + delay_ms;
    if (dst->stim[slot].t0 == t_on) { *scheduled = 1; return EP_OK; }     // already scheduled by an earlier poll
    // windows live on integer steps of the destination (reading A16): the first active step must not be in its past
    if (dst->dt > 0.0 && step_index(t_on, dst->dt) < dst->step)
        return fail(EP_ERR_STATE, "ep_couple polled too late: the stimulus would have started in the destination's past");
    dst->stim[slot].t0 = t_on;
    dst->trig_dirty = true;   // (a trigger of dst driving this slot caches its parameters)
    *scheduled = 1;
    return EP_OK;
}

int ep_read_vext(ep_sim* s, double* out) {
    if (!s || !out) return fail(EP_ERR_ARG, "null argument");
    if (!s->bidomain) return fail(EP_ERR_STATE, "not a bidomain sim (ep_mesh_create_bidomain)");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    int rc = check_sim(s);
    if (rc) return rc;
    if (!s->vext_valid && (rc = bidomain_solve(s))) return rc;
    return read_back(s, s->d_vext, out);
}

int ep_bidomain_solver(ep_sim* s, int restart, int max_cycles, double rel_tol) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (!s->bidomain) return fail(EP_ERR_STATE, "not a bidomain sim (ep_mesh_create_bidomain)");
    if (restart < 1 || restart > 63 || max_cycles < 1 || !(rel_tol > 0.0) || !(rel_tol < 1.0))
        return fail(EP_ERR_ARG, "restart in [1, 63], max_cycles >= 1, 0 < rel_tol < 1");
    if (restart != s->bd_restart && s->gm.V) {
        cudaStreamSynchronize(s->stream);
        s->dev_bytes -= s->gm.bytes;
        epk::gmres_free(s->gm);
    }
    s->bd_restart = restart; s->bd_max_cycles = max_cycles; s->bd_tol = rel_tol;
    s->bd_check = std::min(5, restart);
    return EP_OK;
}

int ep_bidomain_stats(ep_sim* s, int64_t* iters_last, int64_t* iters_total, int64_t* solves, double* rel_res_last) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (!s->bidomain) return fail(EP_ERR_STATE, "not a bidomain sim (ep_mesh_create_bidomain)");
    if (iters_last) *iters_last = s->bd_iters_last;
    if (iters_total) *iters_total = s->bd_iters_total;
    if (solves) *solves = s->bd_solves;
    if (rel_res_last) *rel_res_last = s->bd_res_last;
    return EP_OK;
}

int ep_set_time_order(ep_sim* s, int order) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (order != 1 && order != 2) return fail(EP_ERR_ARG, "time order must be 1 or 2");
    if (order == 2 && s->model >= 0 && s->model != EP_MODEL_TP06)
        return fail(EP_ERR_ARG, "the second-order scheme is implemented for the TP06 model only");
    int rc = use_device(s);
    if (rc) return rc;
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    if (order == 2 && !s->d_hist) {
        rc = dev_alloc(s, &s->d_hist, (int64_t)epk::O2_ROWS * s->nc_pad);
        if (rc) return rc;
        EP_CUDA(s, cudaMemset(s->d_hist, 0, sizeof(double) * (size_t)epk::O2_ROWS * s->nc_pad));
    }
    if (order != s->order) drop_graphs(s);
    s->order = order;
    s->o2_have = false;
    return EP_OK;
}

int ep_mean_vm(ep_sim* s, double* vbar) {
    if (!s || !vbar) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    epk::launch_weighted_sum(s->nc, s->d_vm[s->cur], s->d_vol, s->d_red, s->d_red + 1024, s->stream);
    s->launches += 2;
    double sum = 0.0;
    EP_CUDA(s, cudaMemcpyAsync(&sum, s->d_red + 1024, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    *vbar = sum / s->vol_total;
    return EP_OK;
}

int ep_check_finite(ep_sim* s, int* all_finite) {
    if (!s || !all_finite) return fail(EP_ERR_ARG, "null argument");
    if (s->model < 0) return fail(EP_ERR_STATE, "no state: call ep_state_init first");
    int rc = use_device(s);
    if (rc) return rc;
    unsigned long long* d_cnt = reinterpret_cast<unsigned long long*>(s->d_red);
    EP_CUDA(s, cudaMemsetAsync(d_cnt, 0, 2 * sizeof(unsigned long long), s->stream));
    epk::launch_state_scan(s->model, s->nc, s->d_vm[s->cur], s->d_y, d_cnt, s->stream);
    s->launches += 1;
    unsigned long long cnt[2] = {0, 0};
    EP_CUDA(s, cudaMemcpyAsync(cnt, d_cnt, sizeof(cnt), cudaMemcpyDeviceToHost, s->stream));
    EP_CUDA(s, cudaStreamSynchronize(s->stream));
    *all_finite = (cnt[0] == 0 && cnt[1] == 0);
    if (!*all_finite) {
        s->sticky = EP_ERR_NUMERIC;
        char msg[200];
        std::snprintf(msg, sizeof msg, "%llu non-finite state values, %llu non-positive concentrations (explicit step unstable? "
                      "see ep_stable_dt)", cnt[0], cnt[1]);
        return fail(EP_ERR_NUMERIC, msg);
    }
    return EP_OK;
}

int ep_math_eval(int fn, int64_t n, const double* x, double* y) {
    if (fn < 0 || fn > 3 || n < 0 || (n > 0 && (!x || !y))) return fail(EP_ERR_ARG, "bad ep_math_eval argument");
    if (n == 0) return EP_OK;
    double *dx = nullptr, *dy = nullptr;
    ep_sim* none = nullptr;
    EP_CUDA(none, cudaMalloc((void**)&dx, sizeof(double) * n));
    if (cudaMalloc((void**)&dy, sizeof(double) * n) != cudaSuccess) { cudaFree(dx); return fail(EP_ERR_NOMEM, "cudaMalloc failed"); }
    cudaError_t e = cudaMemcpy(dx, x, sizeof(double) * n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        epk::launch_math_eval(fn, n, dx, dy, nullptr);
        e = cudaMemcpy(y, dy, sizeof(double) * n, cudaMemcpyDeviceToHost);
    }
    cudaFree(dx); cudaFree(dy);
    if (e != cudaSuccess) return fail(EP_ERR_CUDA, std::string("ep_math_eval: ") + cudaGetErrorString(e));
    return EP_OK;
}

int ep_fp64_rate(double* warp_dfma_per_s) {
    if (!warp_dfma_per_s) return fail(EP_ERR_ARG, "null argument");
    ep_sim* none = nullptr;
    const int64_t len = 592 * 512;
    double* scratch = nullptr;
    EP_CUDA(none, cudaMalloc((void**)&scratch, sizeof(double) * len));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    if (e == cudaSuccess) {
        epk::launch_dfma_rate(scratch, len, 2000, nullptr);   // warm-up: clocks up, code resident
        for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
            cudaEventRecord(e0, nullptr);
            const double n = epk::launch_dfma_rate(scratch, len, 4000, nullptr);   // about 2.3 ms
            cudaEventRecord(e1, nullptr);
            e = cudaEventSynchronize(e1);
            float ms = 0.f;
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
            if (e == cudaSuccess && ms > 0.f) best = std::max(best, n / (ms * 1e-3));
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(scratch);
    if (e != cudaSuccess) return fail(EP_ERR_CUDA, std::string("ep_fp64_rate: ") + cudaGetErrorString(e));
    *warp_dfma_per_s = best;
    return EP_OK;
}

int ep_device_vm(ep_sim* s, void** vm, void** perm) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (vm) *vm = s->d_vm[s->cur];
    if (perm) *perm = s->d_perm;
    return EP_OK;
}

int64_t ep_n_cells(const ep_sim* s) { return s ? s->nc : 0; }
int64_t ep_n_nodes(const ep_sim* s) { return s ? s->nn : 0; }
int64_t ep_step_count(const ep_sim* s) { return s ? s->step : 0; }
double ep_time(const ep_sim* s) { return s ? (double)s->step * s->dt : 0.0; }
int64_t ep_device_bytes(const ep_sim* s) { return s ? s->dev_bytes : 0; }
int64_t ep_launch_count(const ep_sim* s) { return s ? s->launches : 0; }

int ep_profile(ep_sim* s, int enable) {
    if (!s) return fail(EP_ERR_ARG, "null sim handle");
    if (enable) {
        int rc = profile_drain(s);
        if (rc) return rc;
        s->prof_steps = 0.0; s->prof_ms[0] = s->prof_ms[1] = 0.0;
    }
    s->profiling = enable != 0;
    return EP_OK;
}

int ep_profile_read(ep_sim* s, double* out4) {
    if (!s || !out4) return fail(EP_ERR_ARG, "null argument");
    int rc = profile_drain(s);
    if (rc) return rc;
    out4[0] = s->prof_steps; out4[1] = s->prof_ms[0]; out4[2] = s->prof_ms[1]; out4[3] = 0.0;
    return EP_OK;
}

int64_t ep_kernel_bytes(const ep_sim* s, int kernel) {
    if (!s) return 0;
    const int64_t S = s->S > 0 ? s->S : 19;
    if (kernel == 0) return s->star_entries * 12 + s->nn * 8;                 // node table + v_n written
    const int64_t hist = (s->order == 2) ? 2 * 8 * epk::O2_ROWS : 0;           // second order: 8 history rows read + written
    if (kernel == 1) return s->n_owned * (2 * 8 * S + 12 * 12 + 2 + hist) + s->nn * 8;   // states r+w, cell tables, masks, v_n read
    return 0;
}

int64_t ep_step_bytes(const ep_sim* s) {
    if (!s) return 0;
    const int64_t S = s->S > 0 ? s->S : 19;
    // state read + write, cell tables (12 f64 + 12 i32), node table (f64 + i32 per star entry),
    // node values written once and read once, cell type + stimulus mask.  Gathers are assumed cache hits.
    const int64_t hist = (s->order == 2) ? 2 * 8 * epk::O2_ROWS : 0;
    return s->n_owned * (2 * 8 * S + 12 * 12 + 2 + hist) + s->star_entries * 12 + s->nn * 16;
}

}  // extern "C"
