// ep_oracle_o2.cpp -- CPU ORACLE of the second-order time stepping. TEST INFRASTRUCTURE ONLY.
//
// "The numerical error could be reduced by adopting a second-order Adams-Bashforth scheme for the non-gating
// variables ..., although a modified second order Rush-Larsen scheme [79] would be needed to attain a second order accuracy."
// This file states that scheme for the ten Tusscher-Panfilov model on top of the first-order oracle (it includes
// ep_oracle.cpp for the cell model's currents and gate functions, the mesh and the Fig. 8 operator; nothing of the CUDA path):
//
//   non-gating variables u in {v, Ca_i, Ca_SR, Ca_SS, Na_i, K_i}:   u^{n+1} = u^n + dt (3/2 f^n - 1/2 f^{n-1})      (AB2)
//   gating variables (the 13 of reading B1):   y^{n+1} = y_inf(*) + (y^n - y_inf(*)) exp(-dt / tau(*)),
//       (*) = the arguments of y_inf and tau extrapolated to t^{n+1/2}: v* = 3/2 v^n - 1/2 v^{n-1}, and likewise Ca_SS*, Ca_SR*
//       for fCass and Rbar                                                                  (second-order Rush-Larsen)
//   f^n = the right-hand side of PAPER.md:176 at t^n, diffusion term D_c/(chi C_m) included, stimulus EXCLUDED: I_s is
//       piecewise constant with jumps on step boundaries (eq. (4), reading A16), so dt * I_s^n is its exact integral over the
//       step and is added as such (to v, and to K_i by reading B8); extrapolating it across a jump would cost the order.
//   The first step has no history and is the first-order step of PAPER.md:172-176.
// Reading H1: [79]'s generalised Rush-Larsen scheme extrapolates the COEFFICIENTS a = -1/tau, b = y_inf/tau
// (3/2 a^n - 1/2 a^{n-1}); extrapolating their ARGUMENTS instead differs at O(dt^2), keeps the second order, and needs no
// second evaluation of the rate functions.
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (the library also exports everything ep_oracle.cpp exports).
#include "ep_oracle.cpp"

namespace {

// right-hand sides of the six non-gating variables at (y, t^n): order v, Ca_i, Ca_SR, Ca_SS, Na_i, K_i
void tp06_rhs(const double* y, int type, double dv_diff, double* f) {
    Tp06Currents c;
    tp06_currents(y, type, c);
    const double Ca_i = y[14], Ca_SR = y[15], Ca_SS = y[16];
    const double bi = 1.0 / (1.0 + Buf_c * K_bufc / ((Ca_i + K_bufc) * (Ca_i + K_bufc)));
    const double bsr = 1.0 / (1.0 + Buf_sr * K_bufsr / ((Ca_SR + K_bufsr) * (Ca_SR + K_bufsr)));
    const double bss = 1.0 / (1.0 + Buf_ss * K_bufss / ((Ca_SS + K_bufss) * (Ca_SS + K_bufss)));
    f[0] = dv_diff - c.iion;
    f[1] = bi * ((c.Ileak - c.Iup) * V_sr / V_c + c.Ixfer - (c.IbCa + c.IpCa - 2.0 * c.INaCa) * Cap / (2.0 * V_c * F_far));
    f[2] = bsr * (c.Iup - c.Ileak - c.Irel);
    f[3] = bss * (-c.ICaL * Cap / (2.0 * V_ss * F_far) + c.Irel * V_sr / V_ss - c.Ixfer * V_c / V_ss);
    f[4] = -(c.INa + c.IbNa + 3.0 * c.INaK + 3.0 * c.INaCa) * Cap / (V_c * F_far);
    f[5] = -(c.IK1 + c.Ito + c.IKr + c.IKs - 2.0 * c.INaK + c.IpK) * Cap / (V_c * F_far);
}

struct Hist {            // what one cell remembers of t^{n-1}
    double v, CaSS, CaSR, f[6];
};

// One second-order step of one cell.  have = 0: no history yet (first-order step).  hist is updated to t^n either way.
void tp06_step_o2(const double* y, int type, double dt, double istim, double dv_diff, Hist& h, int have, double* yn) {
    double f[6];
    tp06_rhs(y, type, dv_diff, f);
    if (!have) {
        tp06_step(y, type, dt, istim, dv_diff, yn);
    } else {
        const double vs = 1.5 * y[0] - 0.5 * h.v;
        const double CaSSs = 1.5 * y[16] - 0.5 * h.CaSS, CaSRs = 1.5 * y[15] - 0.5 * h.CaSR;
        double inf[13], tau[13];
        tp06_gates(vs, type, CaSSs, CaSRs, inf, tau);
        for (int g = 0; g < 13; ++g) yn[1 + g] = inf[g] + (y[1 + g] - inf[g]) * std::exp(-dt / tau[g]);
        const int idx[6] = {0, 14, 15, 16, 17, 18};
        for (int k = 0; k < 6; ++k) yn[idx[k]] = y[idx[k]] + dt * (1.5 * f[k] - 0.5 * h.f[k]);
        yn[0] -= dt * istim;                                   // exact integral of the stimulus over the step
        yn[18] -= dt * istim * Cap / (V_c * F_far);            // reading B8
    }
    h.v = y[0]; h.CaSS = y[16]; h.CaSR = y[15];
    for (int k = 0; k < 6; ++k) h.f[k] = f[k];
}

struct SimO2 {
    Sim* s = nullptr;
    std::vector<Hist> hist;
    int have = 0;
};

}  // namespace

extern "C" {

// attaches second-order stepping to an oracle sim created by orc_create + orc_state_init(model 0)
void* orc_o2_attach(void* h) {
    SimO2* o = new SimO2();
    o->s = (Sim*)h;
    o->hist.resize(o->s->nc);
    return o;
}
void orc_o2_detach(void* p) { delete (SimO2*)p; }
void orc_o2_reset(void* p) { ((SimO2*)p)->have = 0; }

int orc_o2_step(void* p, int64_t n_steps, double dt) {
    SimO2& o = *(SimO2*)p;
    Sim& s = *o.s;
    if (s.model != 0 || !(dt > 0)) return -3;
    s.dt = dt;
    const int64_t nc = s.nc;
    const double inv_chiCm = 1.0 / (s.chi * s.Cm);
    for (int64_t it = 0; it < n_steps; ++it) {
        const int64_t n = s.step;
        apply_diffusion(s, s.y.data(), s.D.data(), 1);
        bool on[8];
        for (int k = 0; k < 8; ++k) {
            on[k] = false;
            if (!s.stim[k].set) continue;
            const int64_t n_on = step_index(s.stim[k].t0, dt), n_off = step_index(s.stim[k].t0 + s.stim[k].dur, dt);
            on[k] = (n_on <= n && n < n_off);
        }
#pragma omp parallel for schedule(static)
        for (int64_t c = 0; c < nc; ++c) {
            double y[TP06_S], yn[TP06_S];
            for (int k = 0; k < TP06_S; ++k) y[k] = s.y[(size_t)k * nc + c];
            double Is = 0.0;
            for (int k = 0; k < 8; ++k) if (on[k] && s.stim[k].mask[c]) Is += s.stim[k].amp;
            tp06_step_o2(y, s.ctype[c], dt, Is / s.Cm, s.D[c] * inv_chiCm, o.hist[c], o.have, yn);
            for (int k = 0; k < TP06_S; ++k) s.yn[(size_t)k * nc + c] = yn[k];
            if (s.tact[c] < 0.0 && y[0] <= 0.0 && yn[0] > 0.0) s.tact[c] = (double)(n + 1) * dt;
        }
        s.y.swap(s.yn);
        s.step = n + 1;
        o.have = 1;
    }
    return 0;
}

// single cell: n_steps of the second-order scheme from y (no diffusion), stimulus while n_on <= n < n_off
void orc_tp06_run_o2(double* y, int type, double dt, int64_t n_steps, double istim, int64_t n_on, int64_t n_off,
                     double* vtrace) {
    double yn[TP06_S];
    Hist h;
    int have = 0;
    if (vtrace) vtrace[0] = y[0];
    for (int64_t n = 0; n < n_steps; ++n) {
        const double is = (n_on <= n && n < n_off) ? istim : 0.0;
        tp06_step_o2(y, type, dt, is, 0.0, h, have, yn);
        have = 1;
        std::memcpy(y, yn, sizeof(yn));
        if (vtrace) vtrace[n + 1] = y[0];
    }
}
void orc_tp06_rhs(const double* y, int type, double dv_diff, double* f6) { tp06_rhs(y, type, dv_diff, f6); }
// one step with explicit history (pins): hist9 = {v, CaSS, CaSR, f[6]} of t^{n-1}, updated in place
void orc_tp06_step_o2(const double* y, int type, double dt, double istim, double dv_diff, double* hist9, int have, double* yn) {
    Hist h;
    h.v = hist9[0]; h.CaSS = hist9[1]; h.CaSR = hist9[2];
    for (int k = 0; k < 6; ++k) h.f[k] = hist9[3 + k];
    tp06_step_o2(y, type, dt, istim, dv_diff, h, have, yn);
    hist9[0] = h.v; hist9[1] = h.CaSS; hist9[2] = h.CaSR;
    for (int k = 0; k < 6; ++k) hist9[3 + k] = h.f[k];
}

}  // extern "C"
