// Internal declarations of librs (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "rs.h"

constexpr int RS_BRICK = 4;                                // brick edge (points)
constexpr int RS_BRICK_PTS = RS_BRICK * RS_BRICK * RS_BRICK;  // 64 points, one uint64 occupancy mask

struct rs_mesh {
    int64_t np = 0;
    double h = 0.0;
    int max_n = 0;
    int periodic = 0;
    int ordering = RS_ORDER_BRICK;
    int lo[3] = {0, 0, 0};    // lattice index of dense cell (0,0,0) (brick aligned)
    int dims[3] = {0, 0, 0};  // dense bounding lattice (multiples of RS_BRICK for brick order)
    int box[3] = {0, 0, 0};   // logical box size (periodic wrap length); = dims for sphere meshes

    std::vector<int32_t> ijk;         // [np][3] lattice indices, mesh order
    std::vector<int32_t> dense2point; // [dims0*dims1*dims2] -> mesh index or -1

    // brick tables (RS_ORDER_BRICK only).  Brick b holds the in-domain points of the 4x4x4 cell at
    // brick coordinates bcoord[b]; local index p = (lx*4 + ly)*4 + lz; present points are stored
    // contiguously from row boff[b] in increasing p; bmask[b] bit p = point p present.
    int nb[3] = {0, 0, 0};
    int64_t nbricks = 0;
    std::vector<int32_t> cell2brick;  // dense brick grid -> brick id or -1
    std::vector<int32_t> boff;        // [nbricks + 1]
    std::vector<uint64_t> bmask;      // [nbricks]
    std::vector<int32_t> bcoord;      // [nbricks][3]

    // device copies
    bool have_device = false;
    int device = -1;
    int sm_count = 0;
    int32_t *d_map[RS_MAX_FD_ORDER + 1] = {nullptr};  // [np][6n], built lazily per order
    int32_t *d_cell2brick = nullptr;
    int32_t *d_boff = nullptr;
    uint64_t *d_bmask = nullptr;
    int32_t *d_bcoord = nullptr;
    void *d_tiles = nullptr;        // brick-kernel work list (see rs_brick.cu)
    int64_t ntiles = 0;
    int *d_counter = nullptr;       // persistent-kernel work counters
};

void rs_set_error(const std::string &msg);
rs_status rs_fail(rs_status st, const std::string &msg);
#define RS_CUDA_TRY(call)                                                                         \
    do {                                                                                          \
        cudaError_t _e = (call);                                                                  \
        if (_e != cudaSuccess)                                                                    \
            return rs_fail(RS_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(_e));      \
    } while (0)

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

// rs_brick.cu
bool rs_brick_supported(const rs_mesh *m, int n, int ncol);
rs_status rs_brick_prepare(rs_mesh *m);
rs_status rs_launch_brick(const rs_mesh *m, int n, const rs_weights &w, const double *vloc, const double *psi,
                          double *hpsi, int ncol, cudaStream_t st);
int64_t rs_brick_table_bytes(const rs_mesh *m);
