// Host mesh builder: steps a1-a3 of SURVEY.md section 8(a).
//   a1  enumerate the lattice points in the union of closed balls   (PAPER.md:53 sec. II; :354 sec. XII)
//   a2  choose the point enumeration: lexicographic z-rows (default; what the plane-sweep kernel
//       streams) or the paper's 4x4x4 bricks                         (sec. V.A, Fig. 7)
//   a3  neighbour table; outside points map to the zero slot np      (sec. V.A)
// Everything here runs once per geometry on the host; the tables are uploaded once.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

#include "rs_internal.h"

static thread_local std::string g_err;
void rs_set_error(const std::string &msg) { g_err = msg; }
rs_status rs_fail(rs_status st, const std::string &msg)
{
    g_err = msg;
    return st;
}
extern "C" const char *rs_last_error(void) { return g_err.c_str(); }
extern "C" int rs_version(void) { return 100; }

static inline int floor_div(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

static inline size_t dense_index(const rs_mesh *m, int ix, int iy, int iz) { return rs_dense_index(m, ix, iy, iz); }

// Order the in-domain cells of `in` (dense [dims]) and fill ijk / dense2point / brick tables.
static void enumerate_points(rs_mesh *m, const std::vector<uint8_t> &in)
{
    const int nx = m->dims[0], ny = m->dims[1], nz = m->dims[2];
    m->dense2point.assign((size_t)nx * ny * nz, -1);
    m->ijk.clear();
    int64_t count = 0;
    auto push = [&](int ix, int iy, int iz) {
        m->dense2point[dense_index(m, ix, iy, iz)] = (int32_t)count++;
        m->ijk.push_back(m->lo[0] + ix);
        m->ijk.push_back(m->lo[1] + iy);
        m->ijk.push_back(m->lo[2] + iz);
    };
    if (m->ordering == RS_ORDER_LEX) {
        for (int ix = 0; ix < nx; ++ix)
            for (int iy = 0; iy < ny; ++iy)
                for (int iz = 0; iz < nz; ++iz)
                    if (in[dense_index(m, ix, iy, iz)]) push(ix, iy, iz);
        m->np = count;
        return;
    }
    if (m->ordering == RS_ORDER_TILE) {
        // tile columns: the (y, z) plane is cut into 16 x 16 tiles; a tile's points of plane x are consecutive, plane after
        // plane (the order in which the plane-sweep kernel visits the mesh; ordering study)
        constexpr int T = 16;
        for (int ty = 0; ty < ny; ty += T)
            for (int tz = 0; tz < nz; tz += T)
                for (int ix = 0; ix < nx; ++ix)
                    for (int iy = ty; iy < std::min(ny, ty + T); ++iy)
                        for (int iz = tz; iz < std::min(nz, tz + T); ++iz)
                            if (in[dense_index(m, ix, iy, iz)]) push(ix, iy, iz);
        m->np = count;
        return;
    }
    // paper's enumeration: brick after brick, points inside a brick in (x, y, z) order
    const int nb[3] = {m->dims[0] / RS_BRICK, m->dims[1] / RS_BRICK, m->dims[2] / RS_BRICK};
    m->nbricks = 0;
    for (int bx = 0; bx < nb[0]; ++bx)
        for (int by = 0; by < nb[1]; ++by)
            for (int bz = 0; bz < nb[2]; ++bz) {
                const int64_t first = count;
                for (int p = 0; p < RS_BRICK_PTS; ++p) {
                    const int ix = bx * RS_BRICK + (p >> 4), iy = by * RS_BRICK + ((p >> 2) & 3),
                              iz = bz * RS_BRICK + (p & 3);
                    if (in[dense_index(m, ix, iy, iz)]) push(ix, iy, iz);
                }
                if (count > first) ++m->nbricks;
            }
    m->np = count;
}

static rs_status upload(rs_mesh *m)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        m->have_device = false;
        return RS_OK;  // host-only handle: table queries work, compute calls report RS_ERR_CUDA
    }
    RS_CUDA_TRY(cudaGetDevice(&m->device));
    RS_CUDA_TRY(cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, m->device));
    m->have_device = true;
    return RS_OK;
}

static rs_status finish(rs_mesh *m, const std::vector<uint8_t> &in, rs_mesh **out)
{
    enumerate_points(m, in);
    if (m->np <= 0) {
        delete m;
        return rs_fail(RS_ERR_INVALID_ARG, "mesh has no points");
    }
    if (m->np >= (int64_t)1 << 30) {
        delete m;
        return rs_fail(RS_ERR_UNSUPPORTED, "mesh too large for int32 point indices");
    }
    rs_status st = upload(m);
    if (st != RS_OK) {
        rs_mesh_destroy(m);
        return st;
    }
    *out = m;
    return RS_OK;
}

extern "C" rs_status rs_mesh_create_ordered(const double *centers, int nc, double radius, double spacing,
                                            int max_fd_order, rs_ordering ordering, rs_mesh **out)
{
    if (!centers || !out || nc < 1 || !(radius > 0.0) || !(spacing > 0.0) || max_fd_order < 1 ||
        max_fd_order > RS_MAX_FD_ORDER || (ordering != RS_ORDER_BRICK && ordering != RS_ORDER_LEX && ordering != RS_ORDER_TILE))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_mesh_create: bad argument");
    *out = nullptr;
    rs_mesh *m = new (std::nothrow) rs_mesh;
    if (!m) return rs_fail(RS_ERR_ALLOC, "out of host memory");
    m->h = spacing;
    m->max_n = max_fd_order;
    m->ordering = ordering;
    const double R = radius, h = spacing, R2 = R * R;
    for (int a = 0; a < 3; ++a) {
        double mn = centers[a], mx = centers[a];
        for (int A = 1; A < nc; ++A) {
            mn = std::min(mn, centers[3 * A + a]);
            mx = std::max(mx, centers[3 * A + a]);
        }
        int l = (int)std::floor((mn - R) / h) - 1, u = (int)std::ceil((mx + R) / h) + 1;
        l = floor_div(l, RS_BRICK) * RS_BRICK;                 // bricks sit at absolute multiples of 4
        u = (floor_div(u, RS_BRICK) + 1) * RS_BRICK - 1;
        m->lo[a] = l;
        m->dims[a] = u - l + 1;
        m->box[a] = m->dims[a];
    }
    const size_t nbox = (size_t)m->dims[0] * m->dims[1] * m->dims[2];
    if (nbox >= ((size_t)1 << 31)) {
        delete m;
        return rs_fail(RS_ERR_UNSUPPORTED, "bounding lattice too large");
    }
    std::vector<uint8_t> in;
    try {
        in.assign(nbox, 0);
    } catch (...) {
        delete m;
        return rs_fail(RS_ERR_ALLOC, "out of host memory");
    }
    // a1: closed ball |(i,j,k) h - R_A|^2 <= R^2 in fp64 (reading S4), sphere by sphere
    for (int A = 0; A < nc; ++A) {
        const double cx = centers[3 * A], cy = centers[3 * A + 1], cz = centers[3 * A + 2];
        int l[3], u[3];
        for (int a = 0; a < 3; ++a) {
            l[a] = std::max((int)std::floor((centers[3 * A + a] - R) / h) - 1, m->lo[a]);
            u[a] = std::min((int)std::ceil((centers[3 * A + a] + R) / h) + 1, m->lo[a] + m->dims[a] - 1);
        }
        for (int i = l[0]; i <= u[0]; ++i) {
            const double dx = (double)i * h - cx;
            for (int j = l[1]; j <= u[1]; ++j) {
                const double dy = (double)j * h - cy;
                for (int k = l[2]; k <= u[2]; ++k) {
                    const double dz = (double)k * h - cz;
                    const double d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 <= R2) in[dense_index(m, i - m->lo[0], j - m->lo[1], k - m->lo[2])] = 1;
                }
            }
        }
    }
    return finish(m, in, out);
}

extern "C" rs_status rs_mesh_create(const double *centers, int nc, double radius, double spacing, int max_fd_order,
                                    rs_mesh **out)
{
    return rs_mesh_create_ordered(centers, nc, radius, spacing, max_fd_order, RS_ORDER_LEX, out);
}

extern "C" rs_status rs_mesh_create_box(int nx, int ny, int nz, double spacing, int max_fd_order, int periodic,
                                        rs_ordering ordering, rs_mesh **out)
{
    if (!out || nx < 1 || ny < 1 || nz < 1 || !(spacing > 0.0) || max_fd_order < 1 || max_fd_order > RS_MAX_FD_ORDER ||
        (ordering != RS_ORDER_BRICK && ordering != RS_ORDER_LEX && ordering != RS_ORDER_TILE) || (size_t)nx * ny * nz >= ((size_t)1 << 30))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_mesh_create_box: bad argument");
    *out = nullptr;
    rs_mesh *m = new (std::nothrow) rs_mesh;
    if (!m) return rs_fail(RS_ERR_ALLOC, "out of host memory");
    m->h = spacing;
    m->max_n = max_fd_order;
    m->ordering = ordering;
    m->periodic = periodic ? 1 : 0;
    const int n[3] = {nx, ny, nz};
    for (int a = 0; a < 3; ++a) {
        m->lo[a] = 0;
        m->box[a] = n[a];
        m->dims[a] = (n[a] + RS_BRICK - 1) / RS_BRICK * RS_BRICK;
    }
    std::vector<uint8_t> in((size_t)m->dims[0] * m->dims[1] * m->dims[2], 0);
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < ny; ++j)
            for (int k = 0; k < nz; ++k) in[dense_index(m, i, j, k)] = 1;
    return finish(m, in, out);
}

extern "C" rs_status rs_mesh_destroy(rs_mesh *m)
{
    if (!m) return RS_OK;
    if (m->have_device) {
        for (int n = 0; n <= RS_MAX_FD_ORDER; ++n)
            if (m->d_map[n]) cudaFree(m->d_map[n]);
        rs_sweep_free(m);
        cudaFree(m->d_red);
        cudaFree(m->d_ovl);
    }
    delete m;
    return RS_OK;
}

extern "C" int64_t rs_mesh_npoints(const rs_mesh *m) { return m ? m->np : -1; }
extern "C" double rs_mesh_spacing(const rs_mesh *m) { return m ? m->h : 0.0; }
extern "C" int64_t rs_mesh_nbricks(const rs_mesh *m) { return m ? m->nbricks : -1; }

extern "C" rs_status rs_mesh_get_points(const rs_mesh *m, int32_t *ijk_host)
{
    if (!m || !ijk_host) return rs_fail(RS_ERR_INVALID_ARG, "rs_mesh_get_points: null argument");
    std::memcpy(ijk_host, m->ijk.data(), m->ijk.size() * sizeof(int32_t));
    return RS_OK;
}

// a3: map[ip][s], s = axis*2n + 2*(k-1) + (0: +k, 1: -k); np = zero slot.
void rs_build_index_map(const rs_mesh *m, int n, int32_t *map)
{
    const int ns = 6 * n;
    const int32_t zero_slot = (int32_t)m->np;
    for (int64_t ip = 0; ip < m->np; ++ip) {
        int c[3] = {m->ijk[3 * ip] - m->lo[0], m->ijk[3 * ip + 1] - m->lo[1], m->ijk[3 * ip + 2] - m->lo[2]};
        for (int a = 0; a < 3; ++a)
            for (int k = 1; k <= n; ++k)
                for (int sgn = 0; sgn < 2; ++sgn) {
                    int q[3] = {c[0], c[1], c[2]};
                    q[a] += sgn ? -k : k;
                    int32_t v = zero_slot;
                    if (m->periodic) q[a] = ((q[a] % m->box[a]) + m->box[a]) % m->box[a];
                    if (q[a] >= 0 && q[a] < m->dims[a]) {
                        const int32_t j = m->dense2point[dense_index(m, q[0], q[1], q[2])];
                        if (j >= 0) v = j;
                    }
                    map[ip * ns + a * 2 * n + 2 * (k - 1) + sgn] = v;
                }
    }
}

extern "C" rs_status rs_mesh_get_index_map(const rs_mesh *m, int fd_order, int32_t *map_host)
{
    if (!m || !map_host || fd_order < 1 || fd_order > m->max_n)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_mesh_get_index_map: bad argument");
    rs_build_index_map(m, fd_order, map_host);
    return RS_OK;
}

rs_status rs_mesh_device_map(const rs_mesh *cm, int n, const int32_t **d_map)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);  // lazily filled cache inside the handle
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    if (!m->d_map[n]) {
        std::vector<int32_t> map((size_t)m->np * 6 * n);
        rs_build_index_map(m, n, map.data());
        int32_t *d = nullptr;
        RS_CUDA_TRY(cudaMalloc(&d, map.size() * sizeof(int32_t)));
        cudaError_t e = cudaMemcpy(d, map.data(), map.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            cudaFree(d);
            return rs_fail(RS_ERR_CUDA, std::string("map upload: ") + cudaGetErrorString(e));
        }
        m->d_map[n] = d;
    }
    *d_map = m->d_map[n];
    return RS_OK;
}

extern "C" size_t rs_block_bytes(const rs_mesh *m, int block_size, rs_dtype dtype)
{
    if (!m || block_size < 1 || block_size > RS_MAX_BLOCK || (block_size & (block_size - 1))) return 0;
    if (dtype != RS_REAL64 && dtype != RS_COMPLEX128) return 0;
    return (size_t)(m->np + 1) * block_size * (dtype == RS_COMPLEX128 ? 16 : 8);
}
