// Address / undefined-behaviour sanitizer harness for the host preprocessor (paper_2112_12854_b200/csrc/ep_host.cpp) and
// for the oracle's mesh set-up and stepping.  Built and run by tests/test_host_sanitizers.py; not part of the product.
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../paper_2112_12854_b200/csrc/ep_host.h"

extern "C" {
void* orc_create(int64_t, const double*, int64_t, const int32_t*, const double*, const double*, double, double, double, double);
void orc_destroy(void*);
int orc_state_init(void*, int, const uint8_t*, const double*);
int orc_stimulus_set(void*, int, int64_t, const int64_t*, double, double, double);
int orc_trigger_set(void*, int, int64_t, const int64_t*, int, double);
int orc_step(void*, int64_t, double);
double orc_mean_vm(void*);
}

int main() {
    // Kuhn slab nx x ny x nz with a carved corner (so that there are boundary faces inside the box) and a ragged size
    const int nx = 5, ny = 4, nz = 3;
    const double h = 0.3;
    std::vector<double> xyz;
    for (int k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) {
        xyz.push_back(i * h + 0.01 * ((i * 7 + j * 3 + k) % 5)); xyz.push_back(j * h); xyz.push_back(k * h + 0.01 * ((i + j) % 3));
    }
    auto nid = [&](int i, int j, int k) { return (int32_t)(i + (nx + 1) * (j + (ny + 1) * k)); };
    const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    std::vector<int32_t> tets;
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        if (i == nx - 1 && j == ny - 1 && k == nz - 1) continue;   // carved cube
        for (auto& p : perm) {
            int c[3] = {i, j, k};
            tets.push_back(nid(c[0], c[1], c[2]));
            c[p[0]]++; tets.push_back(nid(c[0], c[1], c[2]));
            c[p[1]]++; tets.push_back(nid(c[0], c[1], c[2]));
            tets.push_back(nid(i + 1, j + 1, k + 1));
        }
    }
    const int64_t nn = (int64_t)xyz.size() / 3, nc = (int64_t)tets.size() / 4;
    std::vector<double> fibre(3 * nc), scale(nc);
    for (int64_t c = 0; c < nc; ++c) { fibre[3 * c] = 1.0; fibre[3 * c + 1] = 0.2 * (c % 3); fibre[3 * c + 2] = 0.1; scale[c] = 0.1 + 0.01 * (c % 7); }
    ep::Stencil st; ep::Packed pk; std::string err;
    int rc = ep::build_stencil(nn, xyz.data(), nc, tets.data(), fibre.data(), scale.data(), 1.3, 0.18, 1400.0, 1.0, st, err);
    if (rc) { std::printf("build_stencil failed: %s\n", err.c_str()); return 1; }
    rc = ep::pack(st, xyz.data(), pk, err);
    if (rc) { std::printf("pack failed: %s\n", err.c_str()); return 1; }
    double rowsum = 0.0;
    for (int64_t c = 0; c < nc; ++c) for (int m = 0; m < 8; ++m) rowsum += st.a[8 * c + m];
    // error paths must not leak or overrun either
    std::vector<int32_t> bad(tets); bad[5] = (int32_t)nn + 3;
    ep::Stencil st2;
    if (ep::build_stencil(nn, xyz.data(), nc, bad.data(), nullptr, nullptr, 1.3, 0.18, 1400.0, 1.0, st2, err) == 0) return 2;
    // the oracle: set-up, a stimulus, a trigger, a few steps of each model
    for (int model = 0; model < 2; ++model) {
        void* o = orc_create(nn, xyz.data(), nc, tets.data(), fibre.data(), scale.data(), 1.3, 0.18, 1400.0, 1.0);
        if (!o) return 3;
        std::vector<uint8_t> type(nc);
        for (int64_t c = 0; c < nc; ++c) type[c] = model == 0 ? (uint8_t)(c % 3) : 0;
        orc_state_init(o, model, type.data(), nullptr);
        std::vector<int64_t> ids = {0, 1, 2, 3, 4, 5}, mon = {10, 11}, tgt = {nc - 1, nc - 2};
        orc_stimulus_set(o, 0, (int64_t)ids.size(), ids.data(), -52.0, 0.0, 1.0);
        orc_stimulus_set(o, 1, (int64_t)tgt.size(), tgt.data(), -52.0, 9.0, 0.5);
        orc_trigger_set(o, 0, (int64_t)mon.size(), mon.data(), 1, 0.1);
        orc_step(o, 60, 0.02);
        std::printf("model %d v_bar %.6f\n", model, orc_mean_vm(o));
        orc_destroy(o);
    }
    std::printf("ok nc=%lld nn=%lld slices=%lld rowsum=%.3e\n", (long long)nc, (long long)nn, (long long)pk.n_slices, rowsum);
    return 0;
}
