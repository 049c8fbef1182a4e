// Non-local potential (sec. V.C, eq. 4 at :181):
//   (V_nl phi)(r) = sum_A sum_lm gamma^A_lm(r - R_A) * Integral_{sphere A} gamma^A_lm(r' - R_A) phi(r') dr'
// applied to a block of orbitals in two parts, as the paper does:
//   part 1  the integrals  P[A][lm][j] = h^3 sum_{q in sphere A} gamma[A][q][lm] psi[idx[A][q]][j]   (stored)
//   part 2  hpsi[idx[A][q]][j] += sum_lm gamma[A][q][lm] P[A][lm][j]
// Part 2 writes the same point from two atoms whose spheres overlap: "we divide the atoms in groups whose spheres do
// not overlap. Then, we parallelize over all atoms in each group" (Fig. 11 at :177) -- one launch per
// colour, atoms coloured greedily on the host (two atoms conflict iff they share a mesh point).
// What differs from the paper ("each GPU-thread calculating an integral"): an integral is a cooperative, chunked sum
// (a CTA takes 256 sphere points of one atom for all columns and all lm; the lanes of a point are the block's columns,
// so every psi access is one contiguous row segment), chunk partials are added in a fixed order: deterministic.
// Projector VALUES are an input (pseudopotential data): the caller samples them at the sphere points the library
// publishes (rs_nonlocal_get_sphere).  Readings: closed ball |r - R_A| <= r_c on the mesh; integral =
// lattice sum * h^3; eq. 4 carries no further coefficient.
#include <algorithm>
#include <cmath>
#include <new>

#include "rs_internal.h"

constexpr int NL_CHUNK = 256;      // sphere points per work item
constexpr int NL_THREADS = 256;
constexpr int NL_MAXLM = 16;

struct nl_item {
    int32_t atom, q0, nq;          // sphere points [q0, q0 + nq) of the concatenated arrays
    int32_t first, nchunks;        // the atom's items are [first, first + nchunks)
};

struct rs_nonlocal {
    const rs_mesh *m = nullptr;
    int natoms = 0, nlm = 0, ncolors = 0;
    double rc = 0.0;
    std::vector<int64_t> off;              // [natoms + 1] offsets into idx / gamma (atoms in colour order on the device)
    std::vector<int32_t> idx;              // mesh indices, ascending per atom (host copy, atom order as given)
    std::vector<double> gamma;             // [total][nlm] host copy
    std::vector<int32_t> color;            // [natoms]
    std::vector<char> have;                // projector values set?
    std::vector<nl_item> items;            // sorted by colour
    std::vector<int32_t> color_first;      // [ncolors + 1] item ranges
    // device
    int32_t *d_idx = nullptr;
    double *d_gamma = nullptr, *d_partial = nullptr;
    nl_item *d_items = nullptr;
    bool uploaded = false;
};

namespace {

// part 1: partial[item][lm][c] = sum over the item's points of gamma psi (h^3 applied in part 2)
__global__ void __launch_bounds__(NL_THREADS) nl_project_kernel(const nl_item *__restrict__ items, const int32_t *__restrict__ idx,
                                                               const double *__restrict__ gamma, int nlm, const double *__restrict__ psi,
                                                               int ncol, int tshift, double *__restrict__ partial)
{
    __shared__ double red[NL_THREADS];
    const nl_item it = items[blockIdx.x];
    const int tid = threadIdx.x, c = tid & ((1 << tshift) - 1), prow = tid >> tshift, rpc = NL_THREADS >> tshift;
    double acc[NL_MAXLM];
#pragma unroll
    for (int lm = 0; lm < NL_MAXLM; ++lm) acc[lm] = 0.0;
    if (c < ncol)
        for (int q = it.q0 + prow; q < it.q0 + it.nq; q += rpc) {
            const double v = psi[(size_t)idx[q] * ncol + c];
            const double *g = gamma + (size_t)q * nlm;
#pragma unroll
            for (int lm = 0; lm < NL_MAXLM; ++lm)
                if (lm < nlm) acc[lm] = fma(g[lm], v, acc[lm]);
        }
    for (int lm = 0; lm < nlm; ++lm) {
        __syncthreads();
        red[tid] = acc[lm];
        __syncthreads();
        if (prow == 0 && c < ncol) {
            double s = 0.0;
            for (int r = 0; r < rpc; ++r) s += red[(r << tshift) + c];
            partial[((size_t)blockIdx.x * nlm + lm) * ncol + c] = s;
        }
    }
}

// part 2, one colour: P = h3 * sum of the atom's chunk partials (fixed order), then hpsi += gamma P on the item's points
__global__ void __launch_bounds__(NL_THREADS) nl_scatter_kernel(const nl_item *__restrict__ items, int item0, const int32_t *__restrict__ idx,
                                                               const double *__restrict__ gamma, int nlm, double h3,
                                                               const double *__restrict__ partial, double *__restrict__ hpsi, int ncol,
                                                               int tshift)
{
    __shared__ double P[NL_MAXLM * 128];
    const nl_item it = items[item0 + blockIdx.x];
    const int tid = threadIdx.x, c = tid & ((1 << tshift) - 1), prow = tid >> tshift, rpc = NL_THREADS >> tshift;
    for (int e = tid; e < nlm * ncol; e += NL_THREADS) {
        double s = 0.0;
        for (int k = 0; k < it.nchunks; ++k) s += partial[(size_t)(it.first + k) * nlm * ncol + e];
        P[e] = h3 * s;
    }
    __syncthreads();
    if (c < ncol)
        for (int q = it.q0 + prow; q < it.q0 + it.nq; q += rpc) {
            const double *g = gamma + (size_t)q * nlm;
            double s = 0.0;
            for (int lm = 0; lm < nlm; ++lm) s = fma(g[lm], P[lm * ncol + c], s);
            hpsi[(size_t)idx[q] * ncol + c] += s;
        }
}

int ilog2n(int v)
{
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

}  // namespace

extern "C" rs_status rs_nonlocal_destroy(rs_nonlocal *nl)
{
    if (!nl) return RS_OK;
    cudaFree(nl->d_idx), cudaFree(nl->d_gamma), cudaFree(nl->d_partial), cudaFree(nl->d_items);
    delete nl;
    return RS_OK;
}

extern "C" rs_status rs_nonlocal_create(const rs_mesh *m, const double *centers, int natoms, double rc, int nlm, rs_nonlocal **out)
{
    if (!m || !centers || !out || natoms < 1 || !(rc > 0.0) || nlm < 1 || nlm > NL_MAXLM)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal_create: bad argument");
    *out = nullptr;
    if (m->periodic) return rs_fail(RS_ERR_UNSUPPORTED, "rs_nonlocal_create: periodic meshes are not supported");
    rs_nonlocal *nl = new (std::nothrow) rs_nonlocal;
    if (!nl) return rs_fail(RS_ERR_ALLOC, "out of host memory");
    nl->m = m, nl->natoms = natoms, nl->nlm = nlm, nl->rc = rc;
    const double h = m->h, rc2 = rc * rc;
    nl->off.assign(natoms + 1, 0);
    // sphere membership: closed ball on the lattice, restricted to the mesh; mesh indices ascending per atom
    for (int A = 0; A < natoms; ++A) {
        const double *ctr = centers + 3 * A;
        int lo[3], hi[3];
        for (int a = 0; a < 3; ++a) {
            lo[a] = std::max((int)std::floor((ctr[a] - rc) / h) - 1, m->lo[a]);
            hi[a] = std::min((int)std::ceil((ctr[a] + rc) / h) + 1, m->lo[a] + m->dims[a] - 1);
        }
        const size_t before = nl->idx.size();
        for (int i = lo[0]; i <= hi[0]; ++i)
            for (int j = lo[1]; j <= hi[1]; ++j)
                for (int k = lo[2]; k <= hi[2]; ++k) {
                    const double dx = (double)i * h - ctr[0], dy = (double)j * h - ctr[1], dz = (double)k * h - ctr[2];
                    if (dx * dx + dy * dy + dz * dz > rc2) continue;
                    const int32_t ip = m->dense2point[rs_dense_index(m, i - m->lo[0], j - m->lo[1], k - m->lo[2])];
                    if (ip >= 0) nl->idx.push_back(ip);
                }
        std::sort(nl->idx.begin() + before, nl->idx.end());
        nl->off[A + 1] = (int64_t)nl->idx.size();
    }
    if (nl->idx.size() >= ((size_t)1 << 31)) {
        delete nl;
        return rs_fail(RS_ERR_UNSUPPORTED, "rs_nonlocal_create: too many sphere points");
    }
    nl->gamma.assign(nl->idx.size() * nlm, 0.0);
    nl->have.assign(natoms, 0);
    // colouring: two atoms conflict iff they share a mesh point; greedy, atoms in the given order
    std::vector<std::vector<int32_t>> adj(natoms);
    {
        std::vector<int32_t> owner(m->np, -1), next(nl->idx.size(), -1);   // per point: chain of the atoms that contain it
        for (int A = 0; A < natoms; ++A)
            for (int64_t q = nl->off[A]; q < nl->off[A + 1]; ++q) {
                const int32_t ip = nl->idx[q];
                for (int32_t e = owner[ip]; e >= 0; e = next[e]) {
                    // e is an index into idx of an earlier atom; find that atom
                    const int Bq = (int)(std::upper_bound(nl->off.begin(), nl->off.end(), (int64_t)e) - nl->off.begin()) - 1;
                    if (adj[A].empty() || std::find(adj[A].begin(), adj[A].end(), Bq) == adj[A].end()) {
                        adj[A].push_back(Bq);
                        adj[Bq].push_back(A);
                    }
                }
                next[q] = owner[ip];
                owner[ip] = (int32_t)q;
            }
    }
    nl->color.assign(natoms, -1);
    for (int A = 0; A < natoms; ++A) {
        std::vector<char> used(natoms + 1, 0);
        for (int32_t Bq : adj[A])
            if (nl->color[Bq] >= 0) used[nl->color[Bq]] = 1;
        int c = 0;
        while (used[c]) ++c;
        nl->color[A] = c;
        nl->ncolors = std::max(nl->ncolors, c + 1);
    }
    // work items: chunks of NL_CHUNK sphere points, colour after colour
    nl->color_first.assign(nl->ncolors + 1, 0);
    for (int c = 0; c < nl->ncolors; ++c) {
        nl->color_first[c] = (int32_t)nl->items.size();
        for (int A = 0; A < natoms; ++A) {
            if (nl->color[A] != c) continue;
            const int64_t n = nl->off[A + 1] - nl->off[A];
            const int nch = (int)((n + NL_CHUNK - 1) / NL_CHUNK);
            const int32_t first = (int32_t)nl->items.size();
            for (int k = 0; k < nch; ++k)
                nl->items.push_back({A, (int32_t)(nl->off[A] + (int64_t)k * NL_CHUNK), (int32_t)std::min<int64_t>(NL_CHUNK, n - (int64_t)k * NL_CHUNK),
                                     first, nch});
        }
    }
    nl->color_first[nl->ncolors] = (int32_t)nl->items.size();
    *out = nl;
    return RS_OK;
}

extern "C" int64_t rs_nonlocal_sphere_size(const rs_nonlocal *nl, int atom)
{
    return (nl && atom >= 0 && atom < nl->natoms) ? nl->off[atom + 1] - nl->off[atom] : -1;
}

extern "C" rs_status rs_nonlocal_get_sphere(const rs_nonlocal *nl, int atom, int32_t *mesh_index_host)
{
    if (!nl || !mesh_index_host || atom < 0 || atom >= nl->natoms) return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal_get_sphere: bad argument");
    std::copy(nl->idx.begin() + nl->off[atom], nl->idx.begin() + nl->off[atom + 1], mesh_index_host);
    return RS_OK;
}

extern "C" rs_status rs_nonlocal_set_projectors(rs_nonlocal *nl, int atom, const double *gamma_host)
{
    if (!nl || !gamma_host || atom < 0 || atom >= nl->natoms) return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal_set_projectors: bad argument");
    std::copy(gamma_host, gamma_host + (nl->off[atom + 1] - nl->off[atom]) * nl->nlm, nl->gamma.begin() + nl->off[atom] * nl->nlm);
    nl->have[atom] = 1;
    nl->uploaded = false;
    return RS_OK;
}

extern "C" int rs_nonlocal_ncolors(const rs_nonlocal *nl) { return nl ? nl->ncolors : -1; }

extern "C" rs_status rs_nonlocal_get_colors(const rs_nonlocal *nl, int32_t *color_host)
{
    if (!nl || !color_host) return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal_get_colors: null argument");
    std::copy(nl->color.begin(), nl->color.end(), color_host);
    return RS_OK;
}

// Upload the tables (once the projector values of every atom are set); rs_nonlocal_apply calls it lazily.
extern "C" rs_status rs_nonlocal_prepare(rs_nonlocal *nl)
{
    if (!nl) return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal_prepare: null argument");
    if (!nl->m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    for (char hv : nl->have)
        if (!hv) return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal: projector values of some atom were never set");
    if (nl->uploaded) return RS_OK;
    if (!nl->d_idx) {
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_idx, std::max<size_t>(16, nl->idx.size() * sizeof(int32_t))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_gamma, std::max<size_t>(16, nl->gamma.size() * sizeof(double))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_items, std::max<size_t>(16, nl->items.size() * sizeof(nl_item))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_partial, std::max<size_t>(16, nl->items.size() * (size_t)nl->nlm * 128 * sizeof(double))));
        RS_CUDA_TRY(cudaMemcpy(nl->d_idx, nl->idx.data(), nl->idx.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
        RS_CUDA_TRY(cudaMemcpy(nl->d_items, nl->items.data(), nl->items.size() * sizeof(nl_item), cudaMemcpyHostToDevice));
    }
    RS_CUDA_TRY(cudaMemcpy(nl->d_gamma, nl->gamma.data(), nl->gamma.size() * sizeof(double), cudaMemcpyHostToDevice));
    nl->uploaded = true;
    return RS_OK;
}

extern "C" rs_status rs_nonlocal_apply(rs_nonlocal *nl, const void *psi, void *hpsi, int nst, rs_dtype dtype, void *stream)
{
    if (!nl || !psi || !hpsi || psi == hpsi || nst < 1 || nst > RS_MAX_BLOCK || (nst & (nst - 1)) ||
        (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal_apply: bad argument");
    rs_status rc = rs_nonlocal_prepare(nl);
    if (rc != RS_OK) return rc;
    if (nl->items.empty()) return RS_OK;
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);   // gamma is real: a complex block is 2 nst independent real columns
    const int tshift = ilog2n(ncol);
    cudaStream_t st = (cudaStream_t)stream;
    nl_project_kernel<<<(unsigned)nl->items.size(), NL_THREADS, 0, st>>>(nl->d_items, nl->d_idx, nl->d_gamma, nl->nlm, (const double *)psi,
                                                                        ncol, tshift, nl->d_partial);
    RS_CUDA_TRY(cudaGetLastError());
    const double h3 = nl->m->h * nl->m->h * nl->m->h;
    for (int c = 0; c < nl->ncolors; ++c) {
        const int n = nl->color_first[c + 1] - nl->color_first[c];
        if (n <= 0) continue;
        nl_scatter_kernel<<<(unsigned)n, NL_THREADS, 0, st>>>(nl->d_items, nl->color_first[c], nl->d_idx, nl->d_gamma, nl->nlm, h3,
                                                              nl->d_partial, (double *)hpsi, ncol, tshift);
        RS_CUDA_TRY(cudaGetLastError());
    }
    return RS_OK;
}
