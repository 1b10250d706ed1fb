// ep_oracle2d.cpp -- CPU ORACLE for the two-dimensional (Purkinje) medium. TEST INFRASTRUCTURE ONLY.
//
// Plain, slow fp64 implementation of the explicit monodomain step of arXiv 2112.12854 on a TRIANGULATED SURFACE with
// the Stewart et al. 2009 Purkinje-fibre cell model:
//   * PAPER.md:170  "A similar FV approach is used to discretize the bidomain/monodomain equations over 1D and 2D
//     media": the cell-centred chain of PAPER.md:164-168 (Fig. 8 a->e, eq. (7)-(8)) with triangles for tetrahedra,
//     edges for faces, edge lengths for face areas and triangle areas for cell volumes (a uniform layer thickness
//     cancels between the two);
//   * PAPER.md:126, :174, :256  Stewart model [2] for the Purkinje network: 20 state variables, 13 of them gating
//     variables advanced by Rush-Larsen, the other 7 by forward Euler;
//   * PAPER.md:188-200  the stimulus slots through which communication nodes act (eq. (4)).
// Only tests/ may use this file.  It shares no code, header, table or helper with the CUDA path
// (paper_2112_12854_b200/csrc) nor with oracle/ep_oracle.cpp, and neither includes the other.  No operator
// collapsing, no blocking, no fusion: one loop per panel of Fig. 8.  Readings: A1..A18 as in
// three dimensions, plus
//   D1  edge value v_e = mean of the two nodal values at the edge's end points (the 2D "face centroid" value);
//   D2  a surface embedded in 3D: every cell gradient lies in its own triangle's plane; neighbouring gradients are
//       averaged as 3D vectors; the flux through an edge uses the in-plane outward edge normal of cell c1 (the lower
//       cell id), so it is single-valued and the scheme conservative; on a flat mesh nothing of this matters;
//   D3  M_c = scale [sigma_t I + (sigma_l - sigma_t) f f^T] as in 3D (fibre and sheet-fibre directions
//       with their own conductivities; Table 2 :271 uses the isotropic case for the Purkinje network);
//   B12 Stewart's 13 Rush-Larsen variables are its 13 Hodgkin-Huxley gates y, xr1, xr2, xs, m, h, j, d, f, f2, fCass,
//       s, r; the ryanodine-receptor variable R' is then one of the 7 forward-Euler states (13 + 7 = 20);
//   B13 equations and constants of the Stewart model are restated from the published model (DESIGN.md Appendix C):
//       ten Tusscher-Panfilov 2006 with the hyperpolarisation-activated current I_f (gate y), the sustained current
//       I_sus, a time-independent I_K1, its own I_to kinetics and its own conductances.
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC.  OpenMP loops are over independent cells / nodes / edges.
//
// Pins: tests/test_oracle2d_*.py (uniform field, conservation, linear-field exactness, Gauss-Green identity, cosine-mode
// decay rate, dense brute force, hand-computed gate / current values, reversal potentials, ion-conservation identities,
// Rush-Larsen closed form, automaticity and the paper's "plateau of about 250 ms").

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// ---------------------------------------------------------------------------------------------------------
// Stewart-Aslanidi-Noble-Noble-Boyett-Zhang 2009 human Purkinje-fibre cell (PAPER.md:126 ref [2]).
// Units: mV, ms, mM, currents uA/uF (= pA/pF), conductances nS/pF.
// State order: 0 V, 1 y, 2 xr1, 3 xr2, 4 xs, 5 m, 6 h, 7 j, 8 d, 9 f, 10 f2, 11 fCass, 12 s, 13 r, 14 R',
//              15 Ca_i, 16 Ca_SR, 17 Ca_SS, 18 Na_i, 19 K_i.
namespace stw {
const int S = 20;
const double R_gas = 8314.472, T_abs = 310.0, F_far = 96485.3415;
const double RTF = R_gas * T_abs / F_far;
const double K_o = 5.4, Ca_o = 2.0, Na_o = 140.0;
const double V_c = 0.016404, V_sr = 0.001094, V_ss = 0.00005468, Cap = 0.185;
const double g_fNa = 0.0145654, g_fK = 0.0234346;
const double g_K1 = 0.065, g_Kr = 0.0918, g_Ks = 0.2352, g_Na = 130.5744, g_bNa = 0.00029, g_CaL = 3.98e-5;
const double g_bCa = 0.000592, g_to = 0.08184, g_sus = 0.0227, g_pCa = 0.1238, K_pCa = 0.0005, g_pK = 0.0146;
const double p_KNa = 0.03;
const double P_NaK = 2.724, K_mK = 1.0, K_mNa = 40.0;
const double K_NaCa = 1000.0, K_sat = 0.1, alp = 2.5, gam = 0.35, Km_Ca = 1.38, Km_Nai = 87.5;
const double k1p = 0.15, k2p = 0.045, k3 = 0.06, k4 = 0.005, EC = 1.5, max_sr = 2.5, min_sr = 1.0;
const double V_rel = 0.102, V_xfer = 0.0038, K_up = 0.00025, V_leak = 0.00036, Vmax_up = 0.006375;
const double Buf_c = 0.2, K_bufc = 0.001, Buf_sr = 10.0, K_bufsr = 0.3, Buf_ss = 0.4, K_bufss = 0.00025;

// initial state of the published model (a point of its spontaneous cycle: the cell is auto-rhythmic, there is no rest)
const double INIT[S] = {-69.1370441635924, 0.0457562667986602, 0.00550281999719088, 0.313213286437995,
                        0.00953708522974789, 0.0417391656294997, 0.190678733735145, 0.238219836154029,
                        0.000287906256206415, 0.989328560287987, 0.995474890442185, 0.999955429598213,
                        0.96386101799501, 0.00103618091196912, 0.991580051907845,
                        0.000101878186157052, 3.10836886659417, 0.000446818714055411, 8.80420286531673,
                        136.781894160227};

inline double sig(double z) { return 1.0 / (1.0 + std::exp(z)); }   // 1/(1+e^z)

// steady states and time constants of the 13 gates, index g = state index - 1 (0 y ... 12 r)
void gates(double v, double Ca_SS, double* inf, double* tau) {
    // y (I_f)
    inf[0] = sig((v + 80.6) / 6.8);
    tau[0] = 4000.0 / (std::exp(-2.9 - 0.04 * v) + std::exp(3.6 + 0.11 * v));
    // xr1, xr2, xs
    inf[1] = sig((-26.0 - v) / 7.0);
    tau[1] = 450.0 * sig((-45.0 - v) / 10.0) * 6.0 * sig((v + 30.0) / 11.5);
    inf[2] = sig((v + 88.0) / 24.0);
    tau[2] = 3.0 * sig((-60.0 - v) / 20.0) * 1.12 * sig((v - 60.0) / 20.0);
    inf[3] = sig((-5.0 - v) / 14.0);
    tau[3] = 1400.0 / std::sqrt(1.0 + std::exp((5.0 - v) / 6.0)) * sig((v - 35.0) / 15.0) + 80.0;
    // m
    { const double s = sig((-56.86 - v) / 9.03); inf[4] = s * s;
      tau[4] = sig((-60.0 - v) / 5.0) * (0.1 * sig((v + 35.0) / 5.0) + 0.1 * sig((v - 50.0) / 200.0)); }
    // h, j (v >= -40 takes the high-voltage branch, reading B7)
    { const double s = sig((v + 71.55) / 7.43); inf[5] = s * s; inf[6] = s * s;
      double ah, bh, aj, bj;
      if (v >= -40.0) {
          ah = 0.0; bh = 0.77 / (0.13 * (1.0 + std::exp(-(v + 10.66) / 11.1)));
          aj = 0.0; bj = 0.6 * std::exp(0.057 * v) / (1.0 + std::exp(-0.1 * (v + 32.0)));
      } else {
          ah = 0.057 * std::exp(-(v + 80.0) / 6.8);
          bh = 2.7 * std::exp(0.079 * v) + 3.1e5 * std::exp(0.3485 * v);
          aj = (-2.5428e4 * std::exp(0.2444 * v) - 6.948e-6 * std::exp(-0.04391 * v)) * (v + 37.78)
               / (1.0 + std::exp(0.311 * (v + 79.23)));
          bj = 0.02424 * std::exp(-0.01052 * v) / (1.0 + std::exp(-0.1378 * (v + 40.14)));
      }
      tau[5] = 1.0 / (ah + bh); tau[6] = 1.0 / (aj + bj); }
    // d, f, f2, fCass
    inf[7] = sig((-8.0 - v) / 7.5);
    tau[7] = (1.4 * sig((-35.0 - v) / 13.0) + 0.25) * (1.4 * sig((v + 5.0) / 5.0)) + sig((50.0 - v) / 20.0);
    inf[8] = sig((v + 20.0) / 7.0);
    tau[8] = 1102.5 * std::exp(-(v + 27.0) * (v + 27.0) / 225.0) + 200.0 * sig((13.0 - v) / 10.0)
             + 180.0 * sig((v + 30.0) / 10.0) + 20.0;
    inf[9] = 0.67 * sig((v + 35.0) / 7.0) + 0.33;
    tau[9] = 562.0 * std::exp(-(v + 27.0) * (v + 27.0) / 240.0) + 31.0 * sig((25.0 - v) / 10.0)
             + 80.0 * sig((v + 30.0) / 10.0);
    { const double q = 1.0 + (Ca_SS / 0.05) * (Ca_SS / 0.05);
      inf[10] = 0.6 / q + 0.4; tau[10] = 80.0 / q + 2.0; }
    // s, r (Purkinje transient outward current)
    inf[11] = sig((v + 27.0) / 13.0);
    tau[11] = 85.0 * std::exp(-(v + 25.0) * (v + 25.0) / 320.0) + 5.0 * sig((v - 40.0) / 5.0) + 42.0;
    inf[12] = sig((20.0 - v) / 13.0);
    tau[12] = 10.45 * std::exp(-(v + 40.0) * (v + 40.0) / 1800.0) + 7.3;
}

struct Currents {
    double IfNa, IfK, IK1, Ito, Isus, IKr, IKs, ICaL, INaK, INa, IbNa, INaCa, IbCa, IpK, IpCa, iion;
    double Irel, Ileak, Iup, Ixfer, dR;
};

void currents(const double* y, Currents& c) {
    const double v = y[0], yf = y[1], xr1 = y[2], xr2 = y[3], xs = y[4], m = y[5], h = y[6], j = y[7];
    const double d = y[8], f = y[9], f2 = y[10], fcass = y[11], s = y[12], r = y[13], Rp = y[14];
    const double Ca_i = y[15], Ca_SR = y[16], Ca_SS = y[17], Na_i = y[18], K_i = y[19];
    const double E_K = RTF * std::log(K_o / K_i);
    const double E_Na = RTF * std::log(Na_o / Na_i);
    const double E_Ks = RTF * std::log((K_o + p_KNa * Na_o) / (K_i + p_KNa * Na_i));
    const double E_Ca = 0.5 * RTF * std::log(Ca_o / Ca_i);
    c.IfNa = yf * g_fNa * (v - E_Na);
    c.IfK = yf * g_fK * (v - E_K);
    c.IK1 = g_K1 * sig(0.1 * (v + 75.44)) * (v - 8.0 - E_K);
    c.Ito = g_to * r * s * (v - E_K);
    c.Isus = g_sus * sig((5.0 - v) / 17.0) * (v - E_K);
    c.IKr = g_Kr * std::sqrt(K_o / 5.4) * xr1 * xr2 * (v - E_K);
    c.IKs = g_Ks * xs * xs * (v - E_Ks);
    {   // x/(e^x - 1) -> 1 - x/2 for |x| < 1e-7 (reading B6)
        const double x = 2.0 * (v - 15.0) / RTF;
        const double ex = std::exp(x);
        double xo;
        if (std::fabs(x) < 1e-7) xo = 1.0 - 0.5 * x; else xo = x / (ex - 1.0);
        c.ICaL = g_CaL * d * f * f2 * fcass * 2.0 * F_far * xo * (0.25 * Ca_SS * ex - Ca_o);
    }
    c.INaK = P_NaK * (K_o / (K_o + K_mK)) * (Na_i / (Na_i + K_mNa))
             / (1.0 + 0.1245 * std::exp(-0.1 * v / RTF) + 0.0353 * std::exp(-v / RTF));
    c.INa = g_Na * m * m * m * h * j * (v - E_Na);
    c.IbNa = g_bNa * (v - E_Na);
    {
        const double e1 = std::exp(gam * v / RTF), e2 = std::exp((gam - 1.0) * v / RTF);
        c.INaCa = K_NaCa * (e1 * Na_i * Na_i * Na_i * Ca_o - e2 * Na_o * Na_o * Na_o * Ca_i * alp)
                  / ((Km_Nai * Km_Nai * Km_Nai + Na_o * Na_o * Na_o) * (Km_Ca + Ca_o) * (1.0 + K_sat * e2));
    }
    c.IbCa = g_bCa * (v - E_Ca);
    c.IpK = g_pK * (v - E_K) / (1.0 + std::exp((25.0 - v) / 5.98));
    c.IpCa = g_pCa * Ca_i / (K_pCa + Ca_i);
    c.iion = c.IK1 + c.Ito + c.Isus + c.IKr + c.IKs + c.ICaL + c.INaK + c.INa + c.IbNa + c.INaCa + c.IbCa + c.IpK
             + c.IpCa + c.IfNa + c.IfK;
    {
        const double kcasr = max_sr - (max_sr - min_sr) / (1.0 + (EC / Ca_SR) * (EC / Ca_SR));
        const double k1 = k1p / kcasr, k2 = k2p * kcasr;
        const double O = k1 * Ca_SS * Ca_SS * Rp / (k3 + k1 * Ca_SS * Ca_SS);
        c.Irel = V_rel * O * (Ca_SR - Ca_SS);
        c.Ileak = V_leak * (Ca_SR - Ca_i);
        c.Iup = Vmax_up / (1.0 + K_up * K_up / (Ca_i * Ca_i));
        c.Ixfer = V_xfer * (Ca_SS - Ca_i);
        c.dR = -k2 * Ca_SS * Rp + k4 * (1.0 - Rp);
    }
}

// One explicit step of one cell, right-hand side at t^n.  dv_diff = D_c/(chi C_m) [mV/ms],
// istim = I_s/C_m [uA/uF].  yn may not alias y.
void step(const double* y, double dt, double istim, double dv_diff, double* yn) {
    Currents c;
    currents(y, c);
    double inf[13], tau[13];
    gates(y[0], y[17], inf, tau);
    for (int g = 0; g < 13; ++g)   // Rush-Larsen, PAPER.md:174 (reading B12)
        yn[1 + g] = inf[g] + (y[1 + g] - inf[g]) * std::exp(-dt / tau[g]);
    const double Ca_i = y[15], Ca_SR = y[16], Ca_SS = y[17];
    const double bi = 1.0 / (1.0 + Buf_c * K_bufc / ((Ca_i + K_bufc) * (Ca_i + K_bufc)));      // reading B3
    const double bsr = 1.0 / (1.0 + Buf_sr * K_bufsr / ((Ca_SR + K_bufsr) * (Ca_SR + K_bufsr)));
    const double bss = 1.0 / (1.0 + Buf_ss * K_bufss / ((Ca_SS + K_bufss) * (Ca_SS + K_bufss)));
    const double dCai = bi * ((c.Ileak - c.Iup) * V_sr / V_c + c.Ixfer
                              - (c.IbCa + c.IpCa - 2.0 * c.INaCa) * Cap / (2.0 * V_c * F_far));
    const double dCaSR = bsr * (c.Iup - c.Ileak - c.Irel);
    const double dCaSS = bss * (-c.ICaL * Cap / (2.0 * V_ss * F_far) + c.Irel * V_sr / V_ss - c.Ixfer * V_c / V_ss);
    const double dNai = -(c.INa + c.IbNa + c.IfNa + 3.0 * c.INaK + 3.0 * c.INaCa) * Cap / (V_c * F_far);
    const double dKi = -(c.IK1 + c.Ito + c.IfK + c.Isus + c.IKr + c.IKs + c.IpK + istim - 2.0 * c.INaK) * Cap / (V_c * F_far);
    yn[14] = y[14] + dt * c.dR;
    yn[15] = Ca_i + dt * dCai;
    yn[16] = Ca_SR + dt * dCaSR;
    yn[17] = Ca_SS + dt * dCaSS;
    yn[18] = y[18] + dt * dNai;
    yn[19] = y[19] + dt * dKi;
    yn[0] = y[0] + dt * (dv_diff - c.iion - istim);   // eq. (7)
}
}  // namespace stw

// ---------------------------------------------------------------------------------------------------------
// Cell-centred finite volumes on a triangulated surface (following :164-168 panel by panel).
struct Vec3 { double x, y, z; };
inline Vec3 operator+(Vec3 a, Vec3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline Vec3 operator-(Vec3 a, Vec3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline Vec3 operator*(double s, Vec3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(Vec3 a, Vec3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline Vec3 cross(Vec3 a, Vec3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double norm(Vec3 a) { return std::sqrt(dot(a, a)); }
struct Sym3 { double xx, xy, xz, yy, yz, zz; };
inline Vec3 mul(const Sym3& m, Vec3 a) {
    return {m.xx * a.x + m.xy * a.y + m.xz * a.z, m.xy * a.x + m.yy * a.y + m.yz * a.z,
            m.xz * a.x + m.yz * a.y + m.zz * a.z};
}

struct Edge {             // interior edge, c1 = lower cell id, normal vector outward of c1
    int64_t c1, c2;
    Vec3 s;               // in-plane outward normal of c1 times the edge length
    double a1, a2;        // interpolation weights of the two cell gradients (reading A6)
    Vec3 e;               // unit vector from c2 to c1 (reading A7)
    double d;             // |x_c1 - x_c2|
    Sym3 M;               // conductivity at the edge (reading A8)
};
struct Stim { std::vector<char> mask; double amp, t0, dur; bool set; };

struct Sim2 {
    int64_t nn = 0, nc = 0;
    std::vector<Vec3> x;
    std::vector<int32_t> tri;          // [nc*3]
    std::vector<Vec3> xc;              // vertex centroids (A1)
    std::vector<double> area;
    std::vector<Vec3> se;              // [nc*3] outward in-plane normal of edge j (opposite vertex j) times its length
    std::vector<Sym3> Mc;
    std::vector<Edge> edges;
    std::vector<int64_t> cell_edge;    // [nc*3] interior edge id or -1 (boundary: no flux, A11)
    std::vector<int64_t> star_ptr, star_cell;
    std::vector<double> star_invd;
    double chi = 0, Cm = 0;
    std::vector<double> y, yn;         // [S][nc]
    std::vector<double> tact;
    Stim stim[8];
    int64_t step = 0;
    double dt = 0;
    bool have_state = false;
    std::vector<double> vn, D, flux;
    std::vector<Vec3> grad;
};

const int EDGE_NODES[3][2] = {{1, 2}, {0, 2}, {0, 1}};   // edge j is opposite vertex j

struct EdgeKey { int32_t a, b; int64_t cell; int j; };

int build(Sim2& s, const double* fibre, const double* scale, double sl, double st) {
    const int64_t nc = s.nc, nn = s.nn;
    s.xc.resize(nc); s.area.resize(nc); s.se.resize(3 * nc); s.Mc.resize(nc);
    for (int64_t c = 0; c < nc; ++c) {
        const int32_t* t = &s.tri[3 * c];
        for (int k = 0; k < 3; ++k) if (t[k] < 0 || t[k] >= nn) return -2;
        const Vec3 p[3] = {s.x[t[0]], s.x[t[1]], s.x[t[2]]};
        s.xc[c] = (1.0 / 3.0) * (p[0] + p[1] + p[2]);
        const Vec3 N = cross(p[1] - p[0], p[2] - p[0]);
        s.area[c] = 0.5 * norm(N);
        if (!(s.area[c] > 0.0)) return -2;
        const Vec3 nu = (1.0 / norm(N)) * N;
        for (int j = 0; j < 3; ++j) {
            const Vec3 a = p[EDGE_NODES[j][0]], b = p[EDGE_NODES[j][1]];
            Vec3 sv = cross(b - a, nu);                       // in the triangle's plane, normal to the edge, length |b-a|
            const Vec3 xm = 0.5 * (a + b);
            if (dot(sv, xm - s.xc[c]) < 0.0) sv = -1.0 * sv;  // outward
            s.se[3 * c + j] = sv;
        }
        double fl = sl, ft = st;
        Vec3 f = {0, 0, 0};
        if (fibre) {
            f = {fibre[3 * c], fibre[3 * c + 1], fibre[3 * c + 2]};
            const double n = norm(f);
            if (!(n > 0.0)) return -2;
            f = (1.0 / n) * f;
        } else {
            ft = fl;
        }
        const double sc = scale ? scale[c] : 1.0;
        const double dl = fl - ft;
        s.Mc[c] = {sc * (ft + dl * f.x * f.x), sc * dl * f.x * f.y, sc * dl * f.x * f.z,
                   sc * (ft + dl * f.y * f.y), sc * dl * f.y * f.z, sc * (ft + dl * f.z * f.z)};
    }
    // edges matched by their sorted node pair
    std::vector<EdgeKey> keys(3 * nc);
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j < 3; ++j) {
            int32_t a = s.tri[3 * c + EDGE_NODES[j][0]], b = s.tri[3 * c + EDGE_NODES[j][1]];
            if (a == b) return -2;
            if (a > b) std::swap(a, b);
            keys[3 * c + j] = {a, b, c, j};
        }
    std::sort(keys.begin(), keys.end(), [](const EdgeKey& p, const EdgeKey& q) {
        if (p.a != q.a) return p.a < q.a;
        if (p.b != q.b) return p.b < q.b;
        return p.cell < q.cell;
    });
    s.cell_edge.assign(3 * nc, -1);
    for (size_t i = 0; i < keys.size();) {
        size_t e = i + 1;
        while (e < keys.size() && keys[e].a == keys[i].a && keys[e].b == keys[i].b) ++e;
        if (e - i > 2) return -2;
        if (e - i == 2) {
            const EdgeKey& k1 = keys[i]; const EdgeKey& k2 = keys[i + 1];     // k1.cell < k2.cell
            Edge f;
            f.c1 = k1.cell; f.c2 = k2.cell;
            f.s = s.se[3 * k1.cell + k1.j];
            const Vec3 xm = 0.5 * (s.x[k1.a] + s.x[k1.b]);
            const double d1 = norm(xm - s.xc[f.c1]), d2 = norm(xm - s.xc[f.c2]);
            f.a1 = d2 / (d1 + d2);
            f.a2 = 1.0 - f.a1;
            const Vec3 dc = s.xc[f.c1] - s.xc[f.c2];
            f.d = norm(dc);
            f.e = (1.0 / f.d) * dc;
            const Sym3 &A = s.Mc[f.c1], &B = s.Mc[f.c2];
            f.M = {f.a1 * A.xx + f.a2 * B.xx, f.a1 * A.xy + f.a2 * B.xy, f.a1 * A.xz + f.a2 * B.xz,
                   f.a1 * A.yy + f.a2 * B.yy, f.a1 * A.yz + f.a2 * B.yz, f.a1 * A.zz + f.a2 * B.zz};
            s.cell_edge[3 * k1.cell + k1.j] = (int64_t)s.edges.size();
            s.cell_edge[3 * k2.cell + k2.j] = (int64_t)s.edges.size();
            s.edges.push_back(f);
        }
        i = e;
    }
    // node stars, ascending cell id
    s.star_ptr.assign(nn + 1, 0);
    for (int64_t c = 0; c < nc; ++c) for (int k = 0; k < 3; ++k) s.star_ptr[s.tri[3 * c + k] + 1]++;
    for (int64_t n = 0; n < nn; ++n) s.star_ptr[n + 1] += s.star_ptr[n];
    s.star_cell.resize(3 * nc); s.star_invd.resize(3 * nc);
    std::vector<int64_t> fill(s.star_ptr.begin(), s.star_ptr.end() - 1);
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < 3; ++k) {
            const int32_t n = s.tri[3 * c + k];
            const int64_t p = fill[n]++;
            s.star_cell[p] = c;
            s.star_invd[p] = 1.0 / norm(s.x[n] - s.xc[c]);     // reading A2
        }
    s.vn.resize(nn); s.D.resize(nc); s.flux.resize(s.edges.size()); s.grad.resize(nc);
    return 0;
}

// panel a->b: v_n = sum_k v_k/d_k / sum_k 1/d_k over the cells sharing node n
void node_values(const Sim2& s, const double* v, double* vn) {
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < s.nn; ++n) {
        double num = 0.0, den = 0.0;
        for (int64_t p = s.star_ptr[n]; p < s.star_ptr[n + 1]; ++p) {
            num += v[s.star_cell[p]] * s.star_invd[p];
            den += s.star_invd[p];
        }
        vn[n] = num / den;
    }
}

// panels b->c->d: edge values (reading D1), then Gauss-Green over the triangle's three edges
void cell_gradients(const Sim2& s, const double* vn, Vec3* grad) {
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < s.nc; ++c) {
        Vec3 g = {0, 0, 0};
        for (int j = 0; j < 3; ++j) {
            const double ve = (vn[s.tri[3 * c + EDGE_NODES[j][0]]] + vn[s.tri[3 * c + EDGE_NODES[j][1]]]) / 2.0;
            g = g + ve * s.se[3 * c + j];
        }
        grad[c] = (1.0 / s.area[c]) * g;
    }
}

// panel d->e and the flux of eq. (7): interpolated gradient, eq. (8) correction, (M_f grad v_f) . n L
void edge_fluxes(const Sim2& s, const double* v, const Vec3* grad, double* flux, int use_corr) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)s.edges.size(); ++i) {
        const Edge& f = s.edges[i];
        const Vec3 gbar = f.a1 * grad[f.c1] + f.a2 * grad[f.c2];
        Vec3 g = gbar;
        if (use_corr) g = gbar + ((v[f.c1] - v[f.c2]) / f.d - dot(gbar, f.e)) * f.e;   // eq. (8)
        flux[i] = dot(mul(f.M, g), f.s);
    }
}

void divergence(const Sim2& s, const double* flux, double* D) {
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < s.nc; ++c) {
        double sum = 0.0;
        for (int j = 0; j < 3; ++j) {
            const int64_t e = s.cell_edge[3 * c + j];
            if (e < 0) continue;                                   // boundary edge: no flux (A11)
            sum += (s.edges[e].c1 == c) ? flux[e] : -flux[e];
        }
        D[c] = 100.0 * sum / s.area[c];                            // mS/cm * mV/mm^2 -> uA/cm^3 (A14)
    }
}

void apply_diffusion(Sim2& s, const double* v, double* D, int use_corr) {
    node_values(s, v, s.vn.data());
    cell_gradients(s, s.vn.data(), s.grad.data());
    edge_fluxes(s, v, s.grad.data(), s.flux.data(), use_corr);
    divergence(s, s.flux.data(), D);
}

inline int64_t step_index(double t, double dt) { return (int64_t)std::ceil(t / dt - 1e-9); }   // reading A16

}  // namespace

extern "C" {

void* orc2_create(int64_t n_nodes, const double* xyz, int64_t n_tris, const int32_t* tris, const double* fibre,
                  const double* scale, double sigma_l, double sigma_t, double chi, double Cm) {
    Sim2* s = new Sim2();
    s->nn = n_nodes; s->nc = n_tris; s->chi = chi; s->Cm = Cm;
    s->x.resize(n_nodes);
    for (int64_t n = 0; n < n_nodes; ++n) s->x[n] = {xyz[3 * n], xyz[3 * n + 1], xyz[3 * n + 2]};
    s->tri.assign(tris, tris + 3 * n_tris);
    for (int k = 0; k < 8; ++k) s->stim[k].set = false;
    if (build(*s, fibre, scale, sigma_l, sigma_t) != 0) { delete s; return nullptr; }
    return s;
}
void orc2_destroy(void* h) { delete (Sim2*)h; }
int64_t orc2_n_edges(void* h) { return (int64_t)((Sim2*)h)->edges.size(); }
void orc2_geometry(void* h, double* area, double* centroids) {
    Sim2& s = *(Sim2*)h;
    for (int64_t c = 0; c < s.nc; ++c) {
        area[c] = s.area[c];
        centroids[3 * c] = s.xc[c].x; centroids[3 * c + 1] = s.xc[c].y; centroids[3 * c + 2] = s.xc[c].z;
    }
}
void orc2_node_values(void* h, const double* v, double* vn) { node_values(*(Sim2*)h, v, vn); }
void orc2_cell_gradients(void* h, const double* v, double* grad) {
    Sim2& s = *(Sim2*)h;
    node_values(s, v, s.vn.data());
    cell_gradients(s, s.vn.data(), s.grad.data());
    for (int64_t c = 0; c < s.nc; ++c) { grad[3 * c] = s.grad[c].x; grad[3 * c + 1] = s.grad[c].y; grad[3 * c + 2] = s.grad[c].z; }
}
// D = div(M grad v) in uA/cm^3; use_corr = 0 drops eq. (8) (test hook)
void orc2_apply_diffusion(void* h, const double* v, double* D, int use_corr) { apply_diffusion(*(Sim2*)h, v, D, use_corr); }

int orc2_state_init(void* h, const double* y0) {
    Sim2& s = *(Sim2*)h;
    const double* src = y0 ? y0 : stw::INIT;
    s.y.resize((size_t)stw::S * s.nc); s.yn.resize((size_t)stw::S * s.nc);
    for (int64_t c = 0; c < s.nc; ++c)
        for (int k = 0; k < stw::S; ++k) s.y[(size_t)k * s.nc + c] = src[k];
    s.tact.assign(s.nc, -1.0);
    s.step = 0; s.dt = 0; s.have_state = true;
    return 0;
}
int orc2_stimulus_set(void* h, int slot, int64_t n, const int64_t* ids, double amp, double t0, double dur) {
    Sim2& s = *(Sim2*)h;
    if (slot < 0 || slot >= 8) return -1;
    Stim& st = s.stim[slot];
    st.mask.assign(s.nc, 0);
    for (int64_t i = 0; i < n; ++i) { if (ids[i] < 0 || ids[i] >= s.nc) return -1; st.mask[ids[i]] = 1; }
    st.amp = amp; st.t0 = t0; st.dur = dur; st.set = (n > 0);
    return 0;
}
int orc2_step(void* h, int64_t n_steps, double dt) {
    Sim2& s = *(Sim2*)h;
    if (!s.have_state || !(dt > 0)) return -3;
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
            double y[stw::S], yn[stw::S];
            for (int k = 0; k < stw::S; ++k) y[k] = s.y[(size_t)k * nc + c];
            double Is = 0.0;
            for (int k = 0; k < 8; ++k) if (on[k] && s.stim[k].mask[c]) Is += s.stim[k].amp;
            stw::step(y, dt, Is / s.Cm, s.D[c] * inv_chiCm, yn);
            for (int k = 0; k < stw::S; ++k) s.yn[(size_t)k * nc + c] = yn[k];
            if (s.tact[c] < 0.0 && y[0] <= 0.0 && yn[0] > 0.0) s.tact[c] = (double)(n + 1) * dt;   // A18
        }
        s.y.swap(s.yn);
        s.step = n + 1;
    }
    return 0;
}
void orc2_get_state(void* h, int var, double* out) { Sim2& s = *(Sim2*)h; std::memcpy(out, &s.y[(size_t)var * s.nc], sizeof(double) * s.nc); }
void orc2_set_state(void* h, int var, const double* in) { Sim2& s = *(Sim2*)h; std::memcpy(&s.y[(size_t)var * s.nc], in, sizeof(double) * s.nc); }
void orc2_activation_times(void* h, double* out) { Sim2& s = *(Sim2*)h; std::memcpy(out, s.tact.data(), sizeof(double) * s.nc); }
double orc2_mean_vm(void* h) {
    Sim2& s = *(Sim2*)h;
    double num = 0.0, den = 0.0;
    for (int64_t c = 0; c < s.nc; ++c) { num += s.area[c] * s.y[c]; den += s.area[c]; }
    return num / den;
}

// ---- single-cell entry points
void orc2_stw_init(double* y) { std::memcpy(y, stw::INIT, sizeof(stw::INIT)); }
void orc2_stw_gates(double v, double Ca_SS, double* inf, double* tau) { stw::gates(v, Ca_SS, inf, tau); }
void orc2_stw_currents(const double* y, double* out21) {
    stw::Currents c; stw::currents(y, c);
    const double a[21] = {c.IfNa, c.IfK, c.IK1, c.Ito, c.Isus, c.IKr, c.IKs, c.ICaL, c.INaK, c.INa, c.IbNa, c.INaCa,
                          c.IbCa, c.IpK, c.IpCa, c.iion, c.Irel, c.Ileak, c.Iup, c.Ixfer, c.dR};
    std::memcpy(out21, a, sizeof(a));
}
void orc2_stw_step(const double* y, double dt, double istim, double dv_diff, double* yn) { stw::step(y, dt, istim, dv_diff, yn); }
// n_steps single-cell steps; stimulus istim (uA/uF) while n_on <= n < n_off; optional v trace [n_steps+1];
// freeze_v != 0 holds v at its initial value (Rush-Larsen closed-form pin)
void orc2_stw_run(double* y, double dt, int64_t n_steps, double istim, int64_t n_on, int64_t n_off, double* vtrace,
                  int freeze_v) {
    double yn[stw::S];
    if (vtrace) vtrace[0] = y[0];
    for (int64_t n = 0; n < n_steps; ++n) {
        const double is = (n_on <= n && n < n_off) ? istim : 0.0;
        stw::step(y, dt, is, 0.0, yn);
        if (freeze_v) yn[0] = y[0];
        std::memcpy(y, yn, sizeof(yn));
        if (vtrace) vtrace[n + 1] = y[0];
    }
}

}  // extern "C"
