// Internal declarations of librs (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <map>
#include <string>
#include <tuple>
#include <vector>

#include "rs.h"

constexpr int RS_BRICK = 4;                                   // brick edge (points)
constexpr int RS_BRICK_PTS = RS_BRICK * RS_BRICK * RS_BRICK;  // 64 points

// ---- plane-sweep kernel tables (rs_sweep.cu) -------------------------------------------------------
// The compact form of the neighbour table ("a compact form of it is used"; reading S15):
// one record per (CTA, step).  A CTA's steps walk through its work pieces; a piece is a 16 x 16 tile of
// the (y, z) plane, a range [xa, xb) of x planes and a 16-column slice of the block; its steps cover
// planes xa-4 .. xb+3 (the first and last 4 only feed the x arms).  A record holds
//   runs[RS_SWEEP_MAXRUN]  {first mesh index, destination slot | npoints << 16}: one copy per run of
//                          consecutive in-domain points of a z-row (consecutive in memory in RS_ORDER_LEX);
//   fill[18 (+2 pad)]      bitmap over the stage's [24][24] slots: slots to clear (lattice point outside the mesh
//                          and the stage buffer does not already hold zeros there);
//   hdr[4]                 {2 bits per warp: 0 no mesh point in the warp's 4 x 8 region, 1 centre-only, 2 full;
//                           bits 16..23: entries of the clear list (0xff: walk the bitmap); bit 31: output plane,
//                           column offset of the slice,  bytes copied (1-D runs),  bytes copied (2-D tensor boxes)};
//   flist[64]              uint16 slots to clear, ascending = the set bits of the bitmap when there are at most 64;
//   cidx[256]              mesh index of the tile's own points (-1: outside the mesh / not an output plane).
#define RS_SWEEP_MAXRUN 64
struct rs_sweep_piece {
    int iy, iz, xa, xb, chunk;   // tile, output planes [xa, xb), column slice
    bool operator==(const rs_sweep_piece &o) const { return iy == o.iy && iz == o.iz && xa == o.xa && xb == o.xb && chunk == o.chunk; }
    bool operator!=(const rs_sweep_piece &o) const { return !(*this == o); }
};
struct rs_sweep_host {
    std::vector<int2> items;                         // per CTA: {first record, number of steps}
    std::vector<std::vector<rs_sweep_piece>> pieces; // per CTA, in execution order
    std::vector<unsigned char> recs;                 // [nrec][rec_bytes]
    int rec_bytes = 0;                               // 736 + 4 per tile point (depends on the kernel shape)
    std::vector<int32_t> rec_cell;                   // per record: tile * nx + x of an output plane, -1 for a halo step
    int64_t nrec = 0;
    std::vector<double> load;                        // modelled load per CTA
    double cost_max = 0.0, cost_mean = 0.0;          // modelled load of the busiest / average CTA
};
// measured cost of the kernel's steps on this mesh (rs_hamiltonian_autotune): replaces the cost model when dealing
struct rs_sweep_costs {
    std::vector<float> full;      // [tiles * nx] mean clocks of an output step of (tile, plane); 0 = not measured
    double halo = 0.0;            // mean clocks of a halo step
    double unit = 0.0;            // mean clocks of an output step (all values are used relative to it)
};
struct rs_sweep_tables {
    bool ok = false;              // false: some plane needs more than RS_SWEEP_MAXRUN runs (use the gather kernel)
    int64_t nitems = 0, nrec = 0, bytes = 0;
    int variant = 0;              // which compiled kernel shape the records were built for
    int2 *d_items = nullptr;
    unsigned char *d_recs = nullptr;
    long long *d_cycles = nullptr;                   // per CTA: clock ticks of the last launch
    long long *d_step_clock = nullptr;               // per record: clock at the end of that step (last launch)
    std::vector<int2> host_items;                    // copies kept for rs_hamiltonian_autotune
    std::vector<int32_t> rec_cell;
    std::vector<int64_t> host_stats;                 // per CTA: {steps, pieces, modelled load x 1000, full warp-steps}
    std::vector<std::vector<rs_sweep_piece>> pieces; // the dealing these tables were built from (refined by rs_hamiltonian_autotune)
};

// encoded tensor maps of one psi buffer (rs_sweep.cu: 6 CUtensorMap of 128 bytes), kept per (pointer, row pitch)
struct rs_sweep_map_cache {
    const double *psi = nullptr;
    int ncol = 0;
    alignas(64) unsigned char bytes[6 * 128];
};

struct rs_mesh {
    int64_t np = 0;
    double h = 0.0;
    int max_n = 0;
    int periodic = 0;
    int ordering = RS_ORDER_LEX;
    int lo[3] = {0, 0, 0};    // lattice index of dense cell (0,0,0)
    int dims[3] = {0, 0, 0};  // dense bounding lattice (multiples of RS_BRICK for brick order)
    int box[3] = {0, 0, 0};   // logical box size (periodic wrap length); = dims for sphere meshes

    std::vector<int32_t> ijk;         // [np][3] lattice indices, mesh order
    std::vector<int32_t> dense2point; // [dims0*dims1*dims2] -> mesh index or -1

    int64_t nbricks = 0;              // RS_ORDER_BRICK: number of non-empty 4x4x4 bricks

    // device copies
    bool have_device = false;
    int device = -1;
    int sm_count = 0;
    int32_t *d_map[RS_MAX_FD_ORDER + 1] = {nullptr};                 // [np][6n], built lazily per order
    std::map<std::pair<int, int>, rs_sweep_tables> sweep;            // (fd_order, ncol) -> tables, built lazily
    std::map<std::pair<int, int>, rs_sweep_costs> sweep_costs;       // measured step costs, if autotuned
    std::map<std::pair<int, int>, std::vector<std::vector<rs_sweep_piece>>> sweep_pieces;   // a refined dealing that replaces the dealt one
    std::vector<rs_sweep_map_cache> map_cache;                       // tensor maps per psi buffer (blocks wider than 16 columns)
    rs_sweep_options opt = {32, 1 << 20, 0, 0, 3, 3};                // rs_mesh_set_sweep_options
    double *d_red = nullptr;                                         // per-CTA partial sums of the block reductions (rs_blas.cu)
    double *d_ovl = nullptr;                                         // per-CTA partial matrices of rs_block_overlap (rs_overlap.cu)
};
constexpr int RS_RED_CTAS = 1184;                                    // at most 8 reduction CTAs per SM

void rs_set_error(const std::string &msg);
rs_status rs_fail(rs_status st, const std::string &msg);
#define RS_CUDA_TRY(call)                                                                         \
    do {                                                                                          \
        cudaError_t _e = (call);                                                                  \
        if (_e != cudaSuccess)                                                                    \
            return rs_fail(RS_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(_e));      \
    } while (0)

static inline size_t rs_dense_index(const rs_mesh *m, int ix, int iy, int iz)
{
    return ((size_t)ix * m->dims[1] + iy) * m->dims[2] + iz;
}

// rs_mesh.cu
void rs_build_index_map(const rs_mesh *m, int n, int32_t *map /*[np][6n]*/);
rs_status rs_mesh_device_map(const rs_mesh *m, int n, const int32_t **d_map);

// rs_kernels.cu
struct rs_weights {
    double w[RS_MAX_FD_ORDER + 1];  // w_k = -0.5 c_k / h^2
};
rs_status rs_launch_pack(const rs_mesh *m, const void *states, int64_t ld, int ist0, int nst_in, int B, void *block,
                         int lanes, cudaStream_t st);
rs_status rs_launch_unpack(const rs_mesh *m, const void *block, int B, int nst_in, void *states, int64_t ld, int ist0,
                           int lanes, cudaStream_t st);
rs_status rs_launch_gather(const rs_mesh *m, int n, const rs_weights &w, const int32_t *d_map, const double *vloc,
                           const double *psi, double *hpsi, int ncol, cudaStream_t st);

// rs_sweep.cu
bool rs_sweep_supported(const rs_mesh *m, int n, int ncol);   // static conditions (ordering, order, width)
bool rs_sweep_usable(const rs_mesh *m, int n, int ncol);      // supported, device present and tables built
rs_status rs_launch_sweep(const rs_mesh *m, int n, const rs_weights &w, const double *vloc, const double *psi,
                          double *hpsi, int ncol, cudaStream_t st);
int64_t rs_sweep_table_bytes(const rs_mesh *m, int n, int ncol);
const char *rs_sweep_variant_name(const rs_mesh *m, int n, int ncol);
void rs_sweep_free(rs_mesh *m);
// host-only construction of the records; false if a plane needs more than RS_SWEEP_MAXRUN runs
bool rs_sweep_build_host(const rs_mesh *m, int n, int ncol, int max_planes, int nctas, rs_sweep_host &out,
                         const rs_sweep_costs *measured = nullptr,
                         const std::vector<std::vector<rs_sweep_piece>> *given_pieces = nullptr);
rs_status rs_sweep_prepare(const rs_mesh *m, int n, int ncol);   // build + upload the tables now
rs_status rs_sweep_autotune(const rs_mesh *m, int n, const rs_weights &w, const double *vloc, const double *psi, double *hpsi,
                            int ncol, cudaStream_t st);

// rs_blas.cu: block operations between orbitals (f1)
rs_status rs_launch_block_reduce(const rs_mesh *m, const double *a, const double *b, const double *eps, int ncol, int lanes,
                                 int nq, int mode, double *out, cudaStream_t st);
rs_status rs_launch_block_axpy(const rs_mesh *m, const double *alpha, const double *x, double *y, int ncol, int lanes,
                               cudaStream_t st);
rs_status rs_reduce_scratch(const rs_mesh *m, double **out);

// rs_overlap.cu: overlap / subspace matrices (f2)
rs_status rs_launch_overlap(const rs_mesh *m, const double *x, const double *y, int cr, int lanes, double *M, cudaStream_t st);
rs_status rs_overlap_scratch(const rs_mesh *m, double **out);
