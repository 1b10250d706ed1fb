// ep_host.cpp -- one-time host preprocessor (see ep_host.h and DESIGN.md section 5).  No CUDA, no oracle code.
#include "ep_host.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

namespace ep {
namespace {

enum { ERR_ARG = -1, ERR_MESH = -2 };

struct V3 {
    double x, y, z;
};
inline V3 sub(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 add(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 scl(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 crs(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double len(V3 a) { return std::sqrt(dot(a, a)); }

struct Tensor {  // symmetric 3x3
    double xx, xy, xz, yy, yz, zz;
};
inline V3 apply(const Tensor& m, V3 a) {
    return {m.xx * a.x + m.xy * a.y + m.xz * a.z, m.xy * a.x + m.yy * a.y + m.yz * a.z,
            m.xz * a.x + m.yz * a.y + m.zz * a.z};
}

// Per-cell geometry.  opp[n] is the OUTWARD area vector of the face opposite local vertex n; the gradient of the
// barycentric function of vertex n is -opp[n]/(3V), so that the Gauss-Green gradient of PAPER.md:164 with
// three-node face means equals sum_n v_n * glam[n] (identity P4).
struct CellGeom {
    V3 xc;
    double vol;
    V3 opp[4];
    V3 glam[4];
    V3 xf[4];
};

struct FaceRec {   // one (cell, local face) record bucketed by its smallest node id
    int32_t b, c;  // the two larger node ids, b < c
    int32_t cell;
    int32_t j;
};

// 21-bit-per-axis Morton key
inline uint64_t spread3(uint64_t v) {
    v &= 0x1fffffULL;
    v = (v | v << 32) & 0x1f00000000ffffULL;
    v = (v | v << 16) & 0x1f0000ff0000ffULL;
    v = (v | v << 8) & 0x100f00f00f00f00fULL;
    v = (v | v << 4) & 0x10c30c30c30c30c3ULL;
    v = (v | v << 2) & 0x1249249249249249ULL;
    return v;
}

void morton_order(const double* p, int64_t n, std::vector<int32_t>& perm) {
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t i = 0; i < n; ++i)
        for (int d = 0; d < 3; ++d) {
            lo[d] = std::min(lo[d], p[3 * i + d]);
            hi[d] = std::max(hi[d], p[3 * i + d]);
        }
    // one isotropic scale so that the curve's cells are cubes
    double ext = 0.0;
    for (int d = 0; d < 3; ++d) ext = std::max(ext, hi[d] - lo[d]);
    const double s = ext > 0.0 ? 2097151.0 / ext : 0.0;
    std::vector<std::pair<uint64_t, int32_t>> key(n);
    for (int64_t i = 0; i < n; ++i) {
        uint64_t q[3];
        for (int d = 0; d < 3; ++d) q[d] = (uint64_t)std::min(2097151.0, std::max(0.0, (p[3 * i + d] - lo[d]) * s));
        key[i] = {spread3(q[0]) | (spread3(q[1]) << 1) | (spread3(q[2]) << 2), (int32_t)i};
    }
    std::sort(key.begin(), key.end());
    perm.resize(n);
    for (int64_t i = 0; i < n; ++i) perm[i] = key[i].second;
}

}  // namespace

int build_stencil(int64_t nn, const double* xyz, int64_t nc, const int32_t* tets, const double* fibre,
                  const double* scale, double sigma_l, double sigma_t, double chi, double Cm, Stencil& out,
                  std::string& err) {
    if (nn <= 0 || nc <= 0 || !xyz || !tets) { err = "null pointer or non-positive mesh size"; return ERR_ARG; }
    if (nn > 2000000000LL || nc > 500000000LL) { err = "mesh too large for int32 device indices"; return ERR_ARG; }
    if (!(sigma_l > 0.0) || !(sigma_t > 0.0) || !(chi > 0.0) || !(Cm > 0.0)) {
        err = "sigma_l, sigma_t, chi and Cm must be positive";
        return ERR_ARG;
    }
    for (int64_t i = 0; i < 3 * nn; ++i)
        if (!std::isfinite(xyz[i])) { err = "non-finite node coordinate"; return ERR_MESH; }
    auto P = [&](int32_t n) { return V3{xyz[3 * (int64_t)n], xyz[3 * (int64_t)n + 1], xyz[3 * (int64_t)n + 2]}; };

    // ---- cell geometry and conductivity tensors
    std::vector<CellGeom> g(nc);
    std::vector<Tensor> M(nc);
    for (int64_t c = 0; c < nc; ++c) {
        const int32_t* t = tets + 4 * c;
        for (int k = 0; k < 4; ++k)
            if (t[k] < 0 || t[k] >= nn) { err = "tet node index out of range"; return ERR_MESH; }
        const V3 p[4] = {P(t[0]), P(t[1]), P(t[2]), P(t[3])};
        CellGeom& G = g[c];
        G.xc = scl(0.25, add(add(p[0], p[1]), add(p[2], p[3])));                 // reading A1: vertex centroid
        const double det = dot(crs(sub(p[1], p[0]), sub(p[2], p[0])), sub(p[3], p[0]));
        G.vol = std::fabs(det) / 6.0;
        if (!(G.vol > 0.0)) { err = "degenerate tetrahedron (zero volume)"; return ERR_MESH; }
        for (int n = 0; n < 4; ++n) {
            const V3 a = p[(n + 1) & 3], b = p[(n + 2) & 3], cc = p[(n + 3) & 3];
            V3 s = scl(0.5, crs(sub(b, a), sub(cc, a)));
            if (dot(s, sub(p[n], a)) > 0.0) s = scl(-1.0, s);                     // opposite vertex lies inside
            G.opp[n] = s;
            G.glam[n] = scl(-1.0 / (3.0 * G.vol), s);
            G.xf[n] = scl(1.0 / 3.0, add(add(a, b), cc));
        }
        double sc = scale ? scale[c] : 1.0;
        if (!std::isfinite(sc) || sc < 0.0) { err = "sigma_scale must be finite and non-negative"; return ERR_ARG; }
        double sl = sigma_l, st = sigma_t;
        V3 f = {0, 0, 0};
        if (fibre) {
            f = {fibre[3 * c], fibre[3 * c + 1], fibre[3 * c + 2]};
            const double n = len(f);
            if (!(n > 0.0) || !std::isfinite(n)) { err = "zero or non-finite fibre vector"; return ERR_MESH; }
            f = scl(1.0 / n, f);
        } else {
            st = sl;
        }
        const double dl = sl - st;   // M_c = scale [sigma_t I + (sigma_l - sigma_t) f f^T], eq. (2)-(3), reading A9
        M[c] = {sc * (st + dl * f.x * f.x), sc * dl * f.x * f.y, sc * dl * f.x * f.z,
                sc * (st + dl * f.y * f.y), sc * dl * f.y * f.z, sc * (st + dl * f.z * f.z)};
    }

    // ---- face matching: bucket the 4*nc (cell, face) records by their smallest node id, match inside the bucket
    out.nn = nn; out.nc = nc;
    out.nbr.assign(4 * nc, -1);
    {
        std::vector<int64_t> ptr(nn + 1, 0);
        auto tri = [&](int64_t c, int j, int32_t* n3) {
            const int32_t* t = tets + 4 * c;
            int m = 0;
            for (int k = 0; k < 4; ++k) if (k != j) n3[m++] = t[k];
            std::sort(n3, n3 + 3);
        };
        for (int64_t c = 0; c < nc; ++c)
            for (int j = 0; j < 4; ++j) { int32_t n3[3]; tri(c, j, n3); ptr[n3[0] + 1]++; }
        for (int64_t n = 0; n < nn; ++n) ptr[n + 1] += ptr[n];
        std::vector<FaceRec> rec(4 * nc);
        std::vector<int64_t> fill(ptr.begin(), ptr.end() - 1);
        for (int64_t c = 0; c < nc; ++c)
            for (int j = 0; j < 4; ++j) {
                int32_t n3[3]; tri(c, j, n3);
                if (n3[0] == n3[1] || n3[1] == n3[2]) { err = "tet with a repeated node"; return ERR_MESH; }
                rec[fill[n3[0]]++] = {n3[1], n3[2], (int32_t)c, j};
            }
        for (int64_t n = 0; n < nn; ++n) {
            FaceRec* lo = rec.data() + ptr[n];
            FaceRec* hi = rec.data() + ptr[n + 1];
            std::sort(lo, hi, [](const FaceRec& p, const FaceRec& q) {
                if (p.b != q.b) return p.b < q.b;
                if (p.c != q.c) return p.c < q.c;
                return p.cell < q.cell;
            });
            for (FaceRec* r = lo; r < hi;) {
                FaceRec* e = r + 1;
                while (e < hi && e->b == r->b && e->c == r->c) ++e;
                if (e - r > 2) { err = "face shared by more than two cells"; return ERR_MESH; }
                if (e - r == 2) {
                    out.nbr[4 * (int64_t)r[0].cell + r[0].j] = r[1].cell;
                    out.nbr[4 * (int64_t)r[1].cell + r[1].j] = r[0].cell;
                }
                r = e;
            }
        }
    }

    // ---- node stars with normalised inverse-distance weights (readings A2, A3)
    out.node_ptr.assign(nn + 1, 0);
    for (int64_t c = 0; c < nc; ++c) for (int k = 0; k < 4; ++k) out.node_ptr[tets[4 * c + k] + 1]++;
    for (int64_t n = 0; n < nn; ++n) out.node_ptr[n + 1] += out.node_ptr[n];
    out.node_cell.resize(4 * nc); out.w.resize(4 * nc);
    {
        std::vector<int64_t> fill(out.node_ptr.begin(), out.node_ptr.end() - 1);
        for (int64_t c = 0; c < nc; ++c)
            for (int k = 0; k < 4; ++k) {
                const int32_t n = tets[4 * c + k];
                const int64_t p = fill[n]++;
                out.node_cell[p] = (int32_t)c;
                out.w[p] = 1.0 / len(sub(P(n), g[c].xc));
            }
        for (int64_t n = 0; n < nn; ++n) {
            double s = 0.0;
            for (int64_t p = out.node_ptr[n]; p < out.node_ptr[n + 1]; ++p) s += out.w[p];
            for (int64_t p = out.node_ptr[n]; p < out.node_ptr[n + 1]; ++p) out.w[p] /= s;
        }
    }

    // ---- per-cell coefficients
    out.node.resize(8 * nc); out.a.assign(8 * nc, 0.0); out.b.assign(4 * nc, 0.0);
    out.centroid.resize(3 * nc);
    out.vol.resize(nc);
    for (int64_t c = 0; c < nc; ++c) {
        const int32_t* t = tets + 4 * c;
        const CellGeom& G = g[c];
        out.vol[c] = G.vol;
        out.centroid[3 * c] = G.xc.x; out.centroid[3 * c + 1] = G.xc.y; out.centroid[3 * c + 2] = G.xc.z;
        int32_t slot[8];
        double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        int ns = 4;
        for (int k = 0; k < 4; ++k) slot[k] = t[k];
        const double unit = 100.0 / (G.vol * chi * Cm);   // mS/cm * mV/mm^2 -> uA/cm^3 (x100), then / (chi Cm)
        for (int j = 0; j < 4; ++j) {
            const int64_t c2 = out.nbr[4 * c + j];
            if (c2 < 0) { out.nbr[4 * c + j] = (int32_t)c; continue; }      // boundary face: zero flux
            const CellGeom& H = g[c2];
            const V3 s = G.opp[j];                                          // outward of c
            const double d1 = len(sub(G.xf[j], G.xc)), d2 = len(sub(G.xf[j], H.xc));
            const double al1 = d2 / (d1 + d2), al2 = d1 / (d1 + d2);        // reading A6
            const Tensor& A = M[c]; const Tensor& B = M[c2];
            const Tensor Mf = {al1 * A.xx + al2 * B.xx, al1 * A.xy + al2 * B.xy, al1 * A.xz + al2 * B.xz,
                               al1 * A.yy + al2 * B.yy, al1 * A.yz + al2 * B.yz, al1 * A.zz + al2 * B.zz};  // A8
            const V3 dc = sub(G.xc, H.xc);
            const double d = len(dc);
            const V3 e = scl(1.0 / d, dc);                                  // from the neighbour to c (reading A7)
            const V3 q = apply(Mf, s);                                      // flux = q . grad v_f  (M symmetric)
            const double qe = dot(q, e);
            const V3 p = sub(q, scl(qe, e));                                // part of q seen by the averaged gradient
            // flux out of c = al1 p.grad v_c + al2 p.grad v_c2 + (qe/d)(v_c - v_c2)          (eq. (8) folded in)
            out.b[4 * c + j] = -unit * qe / d;                              // multiplies (v_c2 - v_c)
            for (int k = 0; k < 4; ++k) a[k] += unit * al1 * dot(p, G.glam[k]);
            const int32_t* t2 = tets + 4 * c2;
            for (int k = 0; k < 4; ++k) {
                int m = 0;
                while (m < ns && slot[m] != t2[k]) ++m;
                if (m == ns) {
                    if (ns == 8) { err = "internal: more than 8 nodes around a cell"; return ERR_MESH; }
                    slot[ns++] = t2[k];
                }
                a[m] += unit * al2 * dot(p, H.glam[k]);
            }
        }
        for (int m = 0; m < 8; ++m) {
            out.node[8 * c + m] = m < ns ? slot[m] : slot[0];
            out.a[8 * c + m] = m < ns ? a[m] : 0.0;
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------------------------------
// Two-dimensional media ("a similar FV approach is used to discretize the bidomain/monodomain equations over
// 1D and 2D media"): triangles for tetrahedra, edges for faces, edge lengths for face areas, triangle areas for cell volumes.
// The chain of PAPER.md:164-168 folds into the same factored form with 3 own + <= 3 opposite nodes and 3 edge neighbours, so
// the tables keep their 8 + 4 width (unused slots: coefficient 0) and the device kernels are the three-dimensional ones.
// Readings D1-D3 of DESIGN.md: edge value = mean of its two nodal values; each cell gradient lies in its own triangle's
// plane, neighbouring gradients are combined as 3D vectors and the flux uses the in-plane outward edge normal of the cell
// being summed; M_c = scale [sigma_t I + (sigma_l - sigma_t) f f^T].
int build_stencil_tri(int64_t nn, const double* xyz, int64_t nc, const int32_t* tris, const double* fibre,
                      const double* scale, double sigma_l, double sigma_t, double chi, double Cm, Stencil& out,
                      std::string& err) {
    if (nn <= 0 || nc <= 0 || !xyz || !tris) { err = "null pointer or non-positive mesh size"; return ERR_ARG; }
    if (nn > 2000000000LL || nc > 500000000LL) { err = "mesh too large for int32 device indices"; return ERR_ARG; }
    if (!(sigma_l > 0.0) || !(sigma_t > 0.0) || !(chi > 0.0) || !(Cm > 0.0)) {
        err = "sigma_l, sigma_t, chi and Cm must be positive";
        return ERR_ARG;
    }
    for (int64_t i = 0; i < 3 * nn; ++i)
        if (!std::isfinite(xyz[i])) { err = "non-finite node coordinate"; return ERR_MESH; }
    auto P = [&](int32_t n) { return V3{xyz[3 * (int64_t)n], xyz[3 * (int64_t)n + 1], xyz[3 * (int64_t)n + 2]}; };
    struct TriGeom { V3 xc; double area; V3 opp[3]; V3 glam[3]; V3 xm[3]; };
    std::vector<TriGeom> g(nc);
    std::vector<Tensor> M(nc);
    for (int64_t c = 0; c < nc; ++c) {
        const int32_t* t = tris + 3 * c;
        for (int k = 0; k < 3; ++k)
            if (t[k] < 0 || t[k] >= nn) { err = "triangle node index out of range"; return ERR_MESH; }
        if (t[0] == t[1] || t[1] == t[2] || t[0] == t[2]) { err = "triangle with a repeated node"; return ERR_MESH; }
        const V3 p[3] = {P(t[0]), P(t[1]), P(t[2])};
        TriGeom& G = g[c];
        G.xc = scl(1.0 / 3.0, add(add(p[0], p[1]), p[2]));
        const V3 N = crs(sub(p[1], p[0]), sub(p[2], p[0]));
        const double n2 = len(N);
        G.area = 0.5 * n2;
        if (!(G.area > 0.0)) { err = "degenerate triangle (zero area)"; return ERR_MESH; }
        const V3 nu = scl(1.0 / n2, N);
        for (int n = 0; n < 3; ++n) {
            const V3 a = p[(n + 1) % 3], b = p[(n + 2) % 3];
            V3 s = crs(sub(b, a), nu);                                   // in-plane normal of the edge opposite vertex n
            if (dot(s, sub(p[n], a)) > 0.0) s = scl(-1.0, s);            // the opposite vertex lies inside
            G.opp[n] = s;
            G.glam[n] = scl(-1.0 / (2.0 * G.area), s);                   // gradient of the barycentric function of vertex n
            G.xm[n] = scl(0.5, add(a, b));
        }
        double sc = scale ? scale[c] : 1.0;
        if (!std::isfinite(sc) || sc < 0.0) { err = "sigma_scale must be finite and non-negative"; return ERR_ARG; }
        double sl = sigma_l, st = sigma_t;
        V3 f = {0, 0, 0};
        if (fibre) {
            f = {fibre[3 * c], fibre[3 * c + 1], fibre[3 * c + 2]};
            const double n = len(f);
            if (!(n > 0.0) || !std::isfinite(n)) { err = "zero or non-finite fibre vector"; return ERR_MESH; }
            f = scl(1.0 / n, f);
        } else {
            st = sl;
        }
        const double dl = sl - st;
        M[c] = {sc * (st + dl * f.x * f.x), sc * dl * f.x * f.y, sc * dl * f.x * f.z,
                sc * (st + dl * f.y * f.y), sc * dl * f.y * f.z, sc * (st + dl * f.z * f.z)};
    }
    // ---- edge matching, bucketed by the smaller node id
    out.nn = nn; out.nc = nc;
    out.nbr.assign(4 * nc, -1);
    {
        struct EdgeRec { int32_t b; int32_t cell; int32_t j; };
        std::vector<int64_t> ptr(nn + 1, 0);
        auto ends = [&](int64_t c, int j, int32_t& a, int32_t& b) {
            a = tris[3 * c + (j + 1) % 3]; b = tris[3 * c + (j + 2) % 3];
            if (a > b) std::swap(a, b);
        };
        for (int64_t c = 0; c < nc; ++c)
            for (int j = 0; j < 3; ++j) { int32_t a, b; ends(c, j, a, b); ptr[a + 1]++; }
        for (int64_t n = 0; n < nn; ++n) ptr[n + 1] += ptr[n];
        std::vector<EdgeRec> rec(3 * nc);
        std::vector<int64_t> fill(ptr.begin(), ptr.end() - 1);
        for (int64_t c = 0; c < nc; ++c)
            for (int j = 0; j < 3; ++j) { int32_t a, b; ends(c, j, a, b); rec[fill[a]++] = {b, (int32_t)c, j}; }
        for (int64_t n = 0; n < nn; ++n) {
            EdgeRec* lo = rec.data() + ptr[n];
            EdgeRec* hi = rec.data() + ptr[n + 1];
            std::sort(lo, hi, [](const EdgeRec& p, const EdgeRec& q) { return p.b != q.b ? p.b < q.b : p.cell < q.cell; });
            for (EdgeRec* r = lo; r < hi;) {
                EdgeRec* e = r + 1;
                while (e < hi && e->b == r->b) ++e;
                if (e - r > 2) { err = "edge shared by more than two triangles"; return ERR_MESH; }
                if (e - r == 2) {
                    out.nbr[4 * (int64_t)r[0].cell + r[0].j] = r[1].cell;
                    out.nbr[4 * (int64_t)r[1].cell + r[1].j] = r[0].cell;
                }
                r = e;
            }
        }
    }
    // ---- node stars with normalised inverse-distance weights
    out.node_ptr.assign(nn + 1, 0);
    for (int64_t c = 0; c < nc; ++c) for (int k = 0; k < 3; ++k) out.node_ptr[tris[3 * c + k] + 1]++;
    for (int64_t n = 0; n < nn; ++n) out.node_ptr[n + 1] += out.node_ptr[n];
    out.node_cell.resize(3 * nc); out.w.resize(3 * nc);
    {
        std::vector<int64_t> fill(out.node_ptr.begin(), out.node_ptr.end() - 1);
        for (int64_t c = 0; c < nc; ++c)
            for (int k = 0; k < 3; ++k) {
                const int32_t n = tris[3 * c + k];
                const int64_t p = fill[n]++;
                out.node_cell[p] = (int32_t)c;
                out.w[p] = 1.0 / len(sub(P(n), g[c].xc));
            }
        for (int64_t n = 0; n < nn; ++n) {
            double s = 0.0;
            for (int64_t p = out.node_ptr[n]; p < out.node_ptr[n + 1]; ++p) s += out.w[p];
            for (int64_t p = out.node_ptr[n]; p < out.node_ptr[n + 1]; ++p) out.w[p] /= s;
        }
    }
    // ---- per-cell coefficients: same algebra as in three dimensions
    out.node.resize(8 * nc); out.a.assign(8 * nc, 0.0); out.b.assign(4 * nc, 0.0);
    out.centroid.resize(3 * nc);
    out.vol.resize(nc);
    for (int64_t c = 0; c < nc; ++c) {
        const int32_t* t = tris + 3 * c;
        const TriGeom& G = g[c];
        out.vol[c] = G.area;
        out.centroid[3 * c] = G.xc.x; out.centroid[3 * c + 1] = G.xc.y; out.centroid[3 * c + 2] = G.xc.z;
        int32_t slot[8];
        double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        int ns = 3;
        for (int k = 0; k < 3; ++k) slot[k] = t[k];
        const double unit = 100.0 / (G.area * chi * Cm);
        out.nbr[4 * c + 3] = (int32_t)c;                                    // fourth neighbour slot is never used
        for (int j = 0; j < 3; ++j) {
            const int64_t c2 = out.nbr[4 * c + j];
            if (c2 < 0) { out.nbr[4 * c + j] = (int32_t)c; continue; }      // boundary edge: zero flux
            const TriGeom& H = g[c2];
            // reading D2: the flux through an edge uses the in-plane edge normal of the LOWER-numbered of its two cells
            // (single-valued flux, conservative on a curved surface); from the other side it is that vector reversed
            V3 s = G.opp[j];
            if (c2 < c) {
                const int32_t ea = t[(j + 1) % 3], eb = t[(j + 2) % 3];
                const int32_t* u2 = tris + 3 * c2;
                int j2 = 0;
                for (int q = 0; q < 3; ++q) {
                    const int32_t fa = u2[(q + 1) % 3], fb = u2[(q + 2) % 3];
                    if ((fa == ea && fb == eb) || (fa == eb && fb == ea)) j2 = q;
                }
                s = scl(-1.0, H.opp[j2]);
            }
            const double d1 = len(sub(G.xm[j], G.xc)), d2 = len(sub(G.xm[j], H.xc));
            const double al1 = d2 / (d1 + d2), al2 = d1 / (d1 + d2);
            const Tensor& A = M[c]; const Tensor& B = M[c2];
            const Tensor Mf = {al1 * A.xx + al2 * B.xx, al1 * A.xy + al2 * B.xy, al1 * A.xz + al2 * B.xz,
                               al1 * A.yy + al2 * B.yy, al1 * A.yz + al2 * B.yz, al1 * A.zz + al2 * B.zz};
            const V3 dc = sub(G.xc, H.xc);
            const double d = len(dc);
            const V3 e = scl(1.0 / d, dc);
            const V3 q = apply(Mf, s);
            const double qe = dot(q, e);
            const V3 p = sub(q, scl(qe, e));
            out.b[4 * c + j] = -unit * qe / d;
            for (int k = 0; k < 3; ++k) a[k] += unit * al1 * dot(p, G.glam[k]);
            const int32_t* t2 = tris + 3 * c2;
            for (int k = 0; k < 3; ++k) {
                int m = 0;
                while (m < ns && slot[m] != t2[k]) ++m;
                if (m == ns) slot[ns++] = t2[k];                            // at most 3 + 3 distinct nodes
                a[m] += unit * al2 * dot(p, H.glam[k]);
            }
        }
        for (int m = 0; m < 8; ++m) {
            out.node[8 * c + m] = m < ns ? slot[m] : slot[0];
            out.a[8 * c + m] = m < ns ? a[m] : 0.0;
        }
    }
    return 0;
}

int pack(const Stencil& st, const double* xyz, Packed& out, std::string& err, int64_t n_owned) {
    (void)err;
    const int64_t nc = st.nc, nn = st.nn;
    out.nc = nc; out.nn = nn;
    morton_order(st.centroid.data(), nc, out.perm_c);
    if (n_owned >= 0 && n_owned < nc)   // shard: owned cells first; each group keeps its Morton order
        std::stable_partition(out.perm_c.begin(), out.perm_c.end(), [&](int32_t c) { return (int64_t)c < n_owned; });
    morton_order(xyz, nn, out.perm_n);
    out.inv_c.resize(nc);
    for (int64_t i = 0; i < nc; ++i) out.inv_c[out.perm_c[i]] = (int32_t)i;
    std::vector<int32_t> inv_n(nn);
    for (int64_t i = 0; i < nn; ++i) inv_n[out.perm_n[i]] = (int32_t)i;

    out.nc_pad = (nc + TILE - 1) / TILE * TILE;
    out.cidx.assign(12 * out.nc_pad, 0);
    out.ccoef.assign(12 * out.nc_pad, 0.0);
    out.vol.assign(out.nc_pad, 0.0);
    out.vol_total = 0.0;
    const int64_t n_weighted = (n_owned >= 0 && n_owned < nc) ? n_owned : nc;
    for (int64_t c = 0; c < n_weighted; ++c) out.vol_total += st.vol[c];
    for (int64_t i = 0; i < nc; ++i) {
        const int64_t c = out.perm_c[i];
        out.vol[i] = c < n_weighted ? st.vol[c] : 0.0;
        for (int m = 0; m < 8; ++m) {
            out.cidx[tile_index(i, m, 12)] = inv_n[st.node[8 * c + m]];
            out.ccoef[tile_index(i, m, 12)] = st.a[8 * c + m];
        }
        for (int j = 0; j < 4; ++j) {
            out.cidx[tile_index(i, 8 + j, 12)] = out.inv_c[st.nbr[4 * c + j]];
            out.ccoef[tile_index(i, 8 + j, 12)] = st.b[4 * c + j];
        }
    }
    // node table: sliced ELL (32 nodes per slice, width = largest valence in the slice)
    out.n_slices = (nn + 31) / 32;
    out.slice_ptr.assign(out.n_slices + 1, 0);
    for (int64_t s = 0; s < out.n_slices; ++s) {
        int64_t wmax = 0;
        for (int64_t i = 32 * s; i < std::min(nn, 32 * (s + 1)); ++i) {
            const int64_t n = out.perm_n[i];
            wmax = std::max(wmax, st.node_ptr[n + 1] - st.node_ptr[n]);
        }
        out.slice_ptr[s + 1] = out.slice_ptr[s] + 32 * wmax;
    }
    out.nidx.assign(out.slice_ptr[out.n_slices], 0);
    out.nw.assign(out.slice_ptr[out.n_slices], 0.0);
    out.star_entries = st.node_ptr[nn];
    std::vector<std::pair<int32_t, double>> tmp;
    for (int64_t i = 0; i < nn; ++i) {
        const int64_t n = out.perm_n[i], s = i / 32, lane = i % 32;
        const int64_t wd = (out.slice_ptr[s + 1] - out.slice_ptr[s]) / 32;
        tmp.clear();
        for (int64_t p = st.node_ptr[n]; p < st.node_ptr[n + 1]; ++p)
            tmp.push_back({out.inv_c[st.node_cell[p]], st.w[p]});
        std::sort(tmp.begin(), tmp.end());
        for (int64_t k = 0; k < wd; ++k) {
            const int64_t at = out.slice_ptr[s] + 32 * k + lane;
            if (k < (int64_t)tmp.size()) { out.nidx[at] = tmp[k].first; out.nw[at] = tmp[k].second; }
            else { out.nidx[at] = tmp.empty() ? 0 : tmp[0].first; out.nw[at] = 0.0; }
        }
    }
    return 0;
}


int shard_plan(int64_t nn, const double* xyz, int64_t nc, const int32_t* tets, int part, int n_parts, ShardPlan& out,
               std::string& err) {
    if (nn <= 0 || nc <= 0 || !xyz || !tets) { err = "null pointer or non-positive mesh size"; return ERR_ARG; }
    if (n_parts < 1 || n_parts > 64 || part < 0 || part >= n_parts) { err = "need 0 <= part < n_parts <= 64"; return ERR_ARG; }
    if (nc < n_parts) { err = "fewer cells than parts"; return ERR_ARG; }
    for (int64_t i = 0; i < 4 * nc; ++i)
        if (tets[i] < 0 || tets[i] >= nn) { err = "tet node index out of range"; return ERR_MESH; }
    // ownership: contiguous ranges of the Morton curve through the cell centroids
    std::vector<double> cen(3 * nc);
    for (int64_t c = 0; c < nc; ++c)
        for (int d = 0; d < 3; ++d) {
            double a = 0.0;
            for (int k = 0; k < 4; ++k) a += xyz[3 * (int64_t)tets[4 * c + k] + d];
            cen[3 * c + d] = 0.25 * a;
        }
    std::vector<int32_t> perm;
    morton_order(cen.data(), nc, perm);
    std::vector<uint8_t> owner(nc);
    for (int64_t i = 0; i < nc; ++i) owner[perm[i]] = (uint8_t)((i * n_parts) / nc);
    // node stars
    std::vector<int64_t> ptr(nn + 1, 0);
    for (int64_t i = 0; i < 4 * nc; ++i) ptr[tets[i] + 1]++;
    for (int64_t n = 0; n < nn; ++n) ptr[n + 1] += ptr[n];
    std::vector<int32_t> star(4 * nc);
    {
        std::vector<int64_t> fill(ptr.begin(), ptr.end() - 1);
        for (int64_t c = 0; c < nc; ++c)
            for (int k = 0; k < 4; ++k) star[fill[tets[4 * c + k]]++] = (int32_t)c;
    }
    // ring1[c]: parts owning a cell that shares a node with c; ring2[c]: the same one node-ring further
    std::vector<uint64_t> node_mask(nn, 0), ring1(nc, 0), ring2(nc, 0);
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < 4; ++k) node_mask[tets[4 * c + k]] |= 1ULL << owner[c];
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < 4; ++k) ring1[c] |= node_mask[tets[4 * c + k]];
    std::fill(node_mask.begin(), node_mask.end(), 0);
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < 4; ++k) node_mask[tets[4 * c + k]] |= ring1[c];
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < 4; ++k) ring2[c] |= node_mask[tets[4 * c + k]];
    // local cells: owned (ascending), then halo (ascending)
    out = ShardPlan();
    out.part = part; out.n_parts = n_parts;
    const uint64_t me = 1ULL << part;
    for (int64_t c = 0; c < nc; ++c) if (owner[c] == part) out.local_cells.push_back(c);
    out.n_owned = (int64_t)out.local_cells.size();
    if (out.n_owned == 0) { err = "a part owns no cells"; return ERR_ARG; }
    for (int64_t c = 0; c < nc; ++c) if (owner[c] != part && (ring2[c] & me)) out.local_cells.push_back(c);
    const int64_t nl = (int64_t)out.local_cells.size();
    std::vector<int32_t> cell_local(nc, -1);
    for (int64_t k = 0; k < nl; ++k) cell_local[out.local_cells[k]] = (int32_t)k;
    // local nodes
    std::vector<int32_t> node_local(nn, -1);
    for (int64_t k = 0; k < nl; ++k)
        for (int j = 0; j < 4; ++j) node_local[tets[4 * out.local_cells[k] + j]] = 0;
    for (int64_t n = 0; n < nn; ++n)
        if (node_local[n] == 0) { node_local[n] = (int32_t)out.local_nodes.size(); out.local_nodes.push_back(n); }
    out.local_tets.resize(4 * nl);
    for (int64_t k = 0; k < nl; ++k)
        for (int j = 0; j < 4; ++j) out.local_tets[4 * k + j] = node_local[tets[4 * out.local_cells[k] + j]];
    // exchange lists: what I receive from q = my halo cells owned by q; what I send to q = my owned cells in q's halo
    out.send_ptr.assign(n_parts + 1, 0); out.recv_ptr.assign(n_parts + 1, 0);
    for (int q = 0; q < n_parts; ++q) {
        if (q != part) {
            for (int64_t k = out.n_owned; k < nl; ++k)
                if (owner[out.local_cells[k]] == q) out.recv_cells.push_back(k);
            const uint64_t qb = 1ULL << q;
            for (int64_t k = 0; k < out.n_owned; ++k)
                if (ring2[out.local_cells[k]] & qb) out.send_cells.push_back(k);
        }
        out.send_ptr[q + 1] = (int64_t)out.send_cells.size();
        out.recv_ptr[q + 1] = (int64_t)out.recv_cells.size();
    }
    return 0;
}

}  // namespace ep
