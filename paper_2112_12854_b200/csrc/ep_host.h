// ep_host.h -- one-time host preprocessor of libep.  Plain C++, no CUDA.
//
// Turns (nodes, tets, fibres, sigma) into the factored, atomic-free gather form of the paper's finite-volume
// diffusion operator (Fig. 8 a->e, eq. (7)-(8)):
//
//     v_n        = sum_{k in star(n)} w_nk v_k                       (cell -> node)
//     dv_diff[c] = sum_{m<8} a_cm v_n[node_cm] + sum_{j<4} b_cj (v[nbr_cj] - v[c])      [mV/ms] = D_c / (chi Cm)
//
// The algebra that collapses steps b->e into the 8 + 4 coefficients is derived in DESIGN.md section 5.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace ep {

// Tile-major device layout of every per-cell table with several rows: cells are grouped in tiles
// of TILE consecutive (Morton-ordered) cells, and the `rows` rows of one tile are contiguous: element (cell i, row k)
// sits at ((i / TILE) * rows + k) * TILE + i % TILE.  One thread block works on one tile, so all its rows are at
// compile-time offsets from one base pointer.
constexpr int64_t TILE = 128;
inline int64_t tile_index(int64_t i, int64_t k, int64_t rows) { return ((i / TILE) * rows + k) * TILE + i % TILE; }

struct Stencil {              // caller numbering
    int64_t nn = 0, nc = 0;
    std::vector<int32_t> node;     // [nc*8] node ids touched by cell c (own 4 first), unused slots = node[c*8]
    std::vector<double> a;         // [nc*8]
    std::vector<int32_t> nbr;      // [nc*4] face-neighbour cell (face j is opposite vertex j); boundary => c itself
    std::vector<double> b;         // [nc*4] (0 on boundary faces: no-flux, reading A11)
    std::vector<int64_t> node_ptr; // [nn+1]
    std::vector<int32_t> node_cell;// [nc*4] ([nc*3] for triangles) star cells, ascending cell id
    std::vector<double> w;         // same length: inverse-distance weights, normalised per node
    std::vector<double> centroid;  // [nc*3]
    std::vector<double> vol;       // [nc] cell volumes, mm^3
};

struct Packed {               // device numbering and device layout
    int64_t nn = 0, nc = 0;
    int64_t nc_pad = 0;            // nc rounded up to a multiple of TILE
    std::vector<int32_t> perm_c;   // [nc] device position -> caller cell id
    std::vector<int32_t> inv_c;    // [nc] caller cell id -> device position
    std::vector<int32_t> perm_n;   // [nn]
    std::vector<int32_t> cidx;     // tile-major, 12 rows: rows 0..7 device node ids, rows 8..11 device neighbour cells
    std::vector<double> ccoef;     // tile-major, 12 rows: rows 0..7 a, rows 8..11 b
    // node table: sliced ELL, slices of 32 nodes, entries of slice s start at slice_ptr[s] (in elements) and are laid
    // out [k][lane] with k < slice_w[s]
    int64_t n_slices = 0;
    std::vector<int64_t> slice_ptr;  // [n_slices+1]
    std::vector<int32_t> nidx;       // device cell ids
    std::vector<double> nw;
    int64_t star_entries = 0;        // sum of node valences (= 4*nc), unpadded
    std::vector<double> vol;         // [nc_pad] cell volumes in device order (0 in the padding)
    double vol_total = 0.0;
};

// Returns 0 or a negative EP_ERR_* code; err receives a message.
int build_stencil(int64_t nn, const double* xyz, int64_t nc, const int32_t* tets, const double* fibre,
                  const double* scale, double sigma_l, double sigma_t, double chi, double Cm, Stencil& out,
                  std::string& err);
// The same for a triangulated surface (tris [nc*3]); the tables keep the 8 + 4 layout, unused slots have coefficient 0.
int build_stencil_tri(int64_t nn, const double* xyz, int64_t nc, const int32_t* tris, const double* fibre,
                      const double* scale, double sigma_l, double sigma_t, double chi, double Cm, Stencil& out,
                      std::string& err);
// n_owned < nc: the first n_owned cells (caller numbering) are put first on the device (Morton order among themselves, then
// the rest in Morton order) and only they carry volume weights -- the layout of a shard (owned cells, then halo cells).
int pack(const Stencil& st, const double* xyz, Packed& out, std::string& err, int64_t n_owned = -1);

// Intra-mesh sharding: the cells are cut into n_parts contiguous ranges of the Morton curve through their
// centroids; part p owns one range and keeps, as halo, every other cell within two node-rings of an owned cell (the reach of
// the stencil: the nodes of a cell and of its face neighbours, and the stars of those nodes).  Per step each
// part needs the new Vm of its halo cells from their owners: one neighbour exchange, no global reduction.
struct ShardPlan {
    int part = 0, n_parts = 1;
    int64_t n_owned = 0;
    std::vector<int64_t> local_cells;   // global cell id of local cell k: owned first (ascending global id), then halo (ascending)
    std::vector<int64_t> local_nodes;   // global node id of local node k (ascending)
    std::vector<int32_t> local_tets;    // [n_local*4], local node ids
    std::vector<int64_t> send_ptr, recv_ptr;     // [n_parts+1]: segment of peer q in send_cells / recv_cells
    std::vector<int64_t> send_cells, recv_cells; // LOCAL cell ids; within a segment ascending global id, so that the segment
                                                 // part p sends to q lists the same cells, in the same order, as q's
                                                 // receive segment from p
};
int shard_plan(int64_t nn, const double* xyz, int64_t nc, const int32_t* tets, int part, int n_parts, ShardPlan& out,
               std::string& err);

}  // namespace ep
