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
// One record per (tile, lattice plane x, tile row r): the compact form of the neighbour table
// ("a compact form of it is used"; reading S15).  The tile covers lattice rows
// y = y0 - n + r, r in [0, TY + 2n), and the z window [z0 - n, z0 + TZ + n).  bit zp of `mask` says
// whether lattice point (x, y0 - n + r, z0 - n + zp) is in the mesh; `off` is the mesh index of the
// first such point (in-domain points of a z-row are consecutive in RS_ORDER_LEX).  Halo rows carry
// only the bits of the tile's own z range (the star has no corners).
struct rs_rowinfo {
    int32_t off;
    int32_t pad;
    uint64_t mask;
};
static_assert(sizeof(rs_rowinfo) == 16, "rowinfo is read as one 16-byte vector");

// One work item: output planes [xa, xb) of tile (y0, z0); `tab` = index of the record of plane
// (xa - n), row 0, in the rowinfo array; records of successive planes follow each other.
struct rs_sweep_item {
    int32_t y0, z0, xa, xb;
    int64_t tab;
};

struct rs_sweep_tables {
    int n = 0, ty = 0, tz = 0;
    int64_t nitems = 0;
    int64_t nrecords = 0;
    rs_sweep_item *d_items = nullptr;
    rs_rowinfo *d_rows = nullptr;
    int64_t active_lanes = 0;   // sum over items of (planes * TY * TZ): dense work incl. masked lanes
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
    std::map<std::tuple<int, int, int>, rs_sweep_tables> sweep;      // (n, TY, TZ) -> tables, built lazily
};

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
bool rs_sweep_supported(const rs_mesh *m, int n, int ncol);
rs_status rs_launch_sweep(const rs_mesh *m, int n, const rs_weights &w, const double *vloc, const double *psi,
                          double *hpsi, int ncol, cudaStream_t st);
int64_t rs_sweep_table_bytes(const rs_mesh *m, int n, int ncol);
const char *rs_sweep_variant_name(const rs_mesh *m, int n, int ncol);
void rs_sweep_free(rs_mesh *m);
// host-only construction of the tables (also used by rs_mesh_get_index_map's self-check in tests)
void rs_sweep_build_host(const rs_mesh *m, int n, int ty, int tz, int max_planes, std::vector<rs_sweep_item> &items,
                         std::vector<rs_rowinfo> &rows, int64_t *active_lanes);
