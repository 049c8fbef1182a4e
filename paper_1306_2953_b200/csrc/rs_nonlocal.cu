// Non-local potential (sec. V.C, eq. 4 at :181):
//   (V_nl phi)(r) = sum_A sum_lm gamma^A_lm(r - R_A) * Integral_{sphere A} gamma^A_lm(r' - R_A) phi(r') dr'
// applied to a block of orbitals in two parts, as the paper does:
//   part 1  the integrals  P[A][lm][j] = h^3 sum_{q in sphere A} gamma[A][q][lm] psi[idx[A][q]][j]   (stored)
//   part 2  hpsi[idx[A][q]][j] += sum_lm gamma[A][q][lm] P[A][lm][j]
// Part 2 as a scatter over atoms writes the same point from two atoms whose spheres overlap; the paper's answer:
// "we divide the atoms in groups whose spheres do not overlap. Then, we parallelize over all atoms in each group"
// (Fig. 11 at :177) -- one launch per colour.  On this machine a launch per colour is the whole cost
// (each is a few hundred CTAs of dependent loads: ~30 us apiece, measured), so part 2 runs the other way round, as a
// GATHER over the union of the spheres: the host lists, for every mesh point inside at least one sphere, the
// (atom, sphere point) pairs that cover it (atoms ascending); one thread per (point, column) adds them up and
// updates hpsi once.  No write conflict, no colours, one launch, every point read and written once, and the sum
// order is fixed.  The greedy colouring (two atoms conflict iff they share a mesh point) is still computed and
// published (rs_nonlocal_get_colors) for callers that scatter by atom themselves.
// Part 1: an integral is a cooperative, chunked sum (a CTA takes 256 sphere points of one atom for all columns and
// all lm; the lanes of a point are the block's columns, so every psi access is one contiguous row segment); a small
// second kernel adds an atom's chunk partials in chunk order and stores P = h^3 * sum: deterministic, no atomics.
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
    int32_t slot;                  // the partial sum this item goes into; >= 0 only on the item that completes it
};

struct rs_nonlocal {
    const rs_mesh *m = nullptr;
    int natoms = 0, nlm = 0, ncolors = 0;
    double rc = 0.0;
    std::vector<int64_t> off;              // [natoms + 1] offsets into idx / gamma
    std::vector<int32_t> idx;              // mesh indices, ascending per atom, atoms concatenated in the given order
    std::vector<double> gamma;             // [total][nlm] host copy
    std::vector<int32_t> color;            // [natoms]
    std::vector<char> have;                // projector values set?
    std::vector<nl_item> items;            // atom after atom
    std::vector<int4> atom_slots;          // per atom with sphere points: (atom, first partial slot, slots, -); set by prepare
    int nctas = 0, nslots = 0;             // part 1: persistent CTAs, partial sums they produce
    // union of the spheres, points ascending: urec[u] = (mesh point, q of the first covering pair, its atom | further
    // pairs << 24, start of the further pairs in uext); a pair = (sphere point q in the concatenated arrays, atom)
    std::vector<int4> urec;
    std::vector<int2> uext;
    // device
    int32_t *d_idx = nullptr;
    int4 *d_atom_slots = nullptr;
    int4 *d_urec = nullptr;
    int2 *d_uext = nullptr;
    double *d_gamma = nullptr, *d_partial = nullptr, *d_P = nullptr;
    nl_item *d_items = nullptr;
    bool uploaded = false;
};

namespace {

template <int VEC> struct nl_vec;
template <> struct nl_vec<1> {
    double x;
    static __device__ __forceinline__ nl_vec ld(const double *p) { return {*p}; }
    static __device__ __forceinline__ nl_vec ldcg(const double *p) { return {__ldcg(p)}; }
    __device__ __forceinline__ void st(double *p) const { *p = x; }
    __device__ __forceinline__ void fma_(double g, nl_vec v) { x = fma(g, v.x, x); }
    __device__ __forceinline__ void add(nl_vec v) { x += v.x; }
    __device__ __forceinline__ void scale(double f) { x *= f; }
    __device__ __forceinline__ void add_shfl_xor(int off) { x += __shfl_xor_sync(0xffffffffu, x, off); }
};
template <> struct nl_vec<2> {
    double x, y;
    static __device__ __forceinline__ nl_vec ld(const double *p)
    {
        const double2 v = *reinterpret_cast<const double2 *>(p);
        return {v.x, v.y};
    }
    static __device__ __forceinline__ nl_vec ldcg(const double *p)
    {
        const double2 v = __ldcg(reinterpret_cast<const double2 *>(p));
        return {v.x, v.y};
    }
    __device__ __forceinline__ void st(double *p) const { *reinterpret_cast<double2 *>(p) = make_double2(x, y); }
    __device__ __forceinline__ void fma_(double g, nl_vec v) { x = fma(g, v.x, x), y = fma(g, v.y, y); }
    __device__ __forceinline__ void add(nl_vec v) { x += v.x, y += v.y; }
    __device__ __forceinline__ void scale(double f) { x *= f, y *= f; }
    __device__ __forceinline__ void add_shfl_xor(int off)
    {
        x += __shfl_xor_sync(0xffffffffu, x, off), y += __shfl_xor_sync(0xffffffffu, y, off);
    }
};

// Programmatic dependent launch: the three kernels of one apply are chained so that the next kernel's CTAs become
// resident while the previous kernel drains and do what does not depend on it (tables, hpsi) before they wait.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;\n" ::: "memory"); }

template <class... KArgs, class... Args>
cudaError_t nl_launch(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, bool dependent, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid), cfg.blockDim = dim3(block), cfg.dynamicSmemBytes = smem, cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr, cfg.numAttrs = dependent ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

constexpr int NL_INFLIGHT = 4;     // points per thread in a unit of part 1
constexpr int nl_cps(int lm) { return lm <= 4 ? 3 : lm <= 9 ? 2 : 1; }   // CTAs of part 1 per SM (registers: lm accumulators)
constexpr int NL_GPT = 4;          // points per thread and batch in part 2
constexpr int NL_GATHER_CPS = 3;   // persistent CTAs of part 2 per SM (80 registers; a 4th only fits with spills: slower)
constexpr int NL_LMG = 2;          // lm values reduced per pass through shared memory

__device__ __forceinline__ void cp_async8(void *dst_smem, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

constexpr int NL_STAGES = 3;
__host__ __device__ constexpr int nl_unit(int lshift) { return NL_INFLIGHT * (NL_THREADS >> lshift) < NL_CHUNK ? NL_INFLIGHT * (NL_THREADS >> lshift) : NL_CHUNK; }
constexpr size_t nl_project_smem(int vec, int nlm, int lshift)
{
    return (size_t)NL_STAGES * (NL_INFLIGHT * NL_THREADS * vec * 8 + nl_unit(lshift) * nlm * 8);
}

// Part 1.  A thread owns VEC adjacent columns of the points prow, prow + rows, ... (L = ncol / VEC lanes per point,
// rows = 256 / L points per pass) and LM accumulators per column.  The access chain item -> index -> psi row is three
// dependent trips to memory, and a sphere is small (~17 chunks): one chunk per CTA leaves the machine waiting on
// latency (measured: 1.9 TB/s).  So the CTAs are persistent (one to three per SM) and walk their chunks in UNITS of
// min(256, 4 rows) points through a three-stage cp.async pipeline: while unit u is summed from shared memory the psi
// rows and projector values of units u+1 and u+2 are in flight and the indices of unit u+3 are being loaded.  A thread
// reads back exactly the psi slots it copied; the projector values of a unit are one contiguous span copied by all.
// Reduction over the points at the end of a chunk: shuffles inside a warp (when a warp holds several points), then
// shared memory across the warps, both in a fixed order -> partial[item][lm][c].
template <int VEC, int LM>
__global__ void __launch_bounds__(NL_THREADS, nl_cps(LM)) nl_project_kernel(const nl_item *__restrict__ items, int nitems, const int32_t *__restrict__ idx,
                                                                  const double *__restrict__ gamma, int nlm, const double *__restrict__ psi,
                                                                  int ncol, int lshift, double *__restrict__ partial)
{
    using V = nl_vec<VEC>;
    extern __shared__ __align__(16) unsigned char nl_smem[];
    __shared__ V red[NL_LMG][NL_THREADS];
    pdl_launch_dependents();
    const int tid = threadIdx.x, L = 1 << lshift, cl = tid & (L - 1), prow = tid >> lshift, rows = NL_THREADS >> lshift;
    const int c = cl * VEC;
    const int sub = nl_unit(lshift);                                       // points per unit
    const int psi_bytes = NL_INFLIGHT * NL_THREADS * VEC * 8, stage_bytes = psi_bytes + sub * nlm * 8;
    const int i0 = (int)((long long)blockIdx.x * nitems / gridDim.x), i1 = (int)((long long)(blockIdx.x + 1) * nitems / gridDim.x);
    struct unit {
        int item, q0, end, slot;                                          // points [q0, min(q0 + sub, end)) of the item; item < 0: none
    };
    auto first_unit = [&](int i) {
        if (i >= i1) return unit{-1, 0, 0, -1};
        const nl_item it = items[i];
        return unit{i, it.q0, it.q0 + it.nq, it.slot};
    };
    auto next = [&](unit u) {
        if (u.item < 0) return u;
        if (u.q0 + sub < u.end) return unit{u.item, u.q0 + sub, u.end, u.slot};
        return first_unit(u.item + 1);
    };
    int ipn[NL_INFLIGHT];
    auto load_idx = [&](unit u) {
        const int n = min(sub, u.end - u.q0);
#pragma unroll
        for (int k = 0; k < NL_INFLIGHT; ++k) ipn[k] = prow + k * rows < n ? idx[u.q0 + prow + k * rows] : -1;
    };
    auto issue = [&](unit u, int stage) {
        unsigned char *sp = nl_smem + (size_t)stage * stage_bytes;
#pragma unroll
        for (int k = 0; k < NL_INFLIGHT; ++k)
            if (ipn[k] >= 0) {
                if (VEC == 2) cp_async16(sp + (size_t)(k * NL_THREADS + tid) * 16, psi + (size_t)ipn[k] * ncol + c);
                else cp_async8(sp + (size_t)(k * NL_THREADS + tid) * 8, psi + (size_t)ipn[k] * ncol + c);
            }
        const int words = min(sub, u.end - u.q0) * nlm;
        const double *src = gamma + (size_t)u.q0 * nlm;
        for (int w = tid; w < words; w += NL_THREADS) cp_async8(sp + psi_bytes + (size_t)w * 8, src + w);
        cp_async_commit();
    };
    V acc[LM];
#pragma unroll
    for (int lm = 0; lm < LM; ++lm) acc[lm] = V{};

    unit d0 = first_unit(i0);
    unit d1 = next(d0), d2 = next(d1);
    load_idx(d0), issue(d0, 0);
    load_idx(d1), issue(d1, 1);
    load_idx(d2);
    unit d3 = next(d2);
    for (int stage = 0; d0.item >= 0; stage = stage + 1 == NL_STAGES ? 0 : stage + 1) {
        cp_async_wait<1>();
        __syncthreads();                 // unit d0 has landed for everybody; everybody is done with the stage d2 goes to
        issue(d2, stage + 2 >= NL_STAGES ? stage + 2 - NL_STAGES : stage + 2);
        load_idx(d3);
        const unsigned char *sp = nl_smem + (size_t)stage * stage_bytes;
        const double *gs = reinterpret_cast<const double *>(sp + psi_bytes);
        const int n = min(sub, d0.end - d0.q0);
#pragma unroll
        for (int k = 0; k < NL_INFLIGHT; ++k) {
            if (prow + k * rows >= n) continue;
            const V v = V::ld(reinterpret_cast<const double *>(sp + (size_t)(k * NL_THREADS + tid) * (VEC * 8)));
            const double *g = gs + (size_t)(prow + k * rows) * nlm;
#pragma unroll
            for (int lm = 0; lm < LM; ++lm)
                if (lm < nlm) acc[lm].fma_(g[lm], v);
        }
        if (d0.q0 + sub >= d0.end && d0.slot >= 0) {   // the CTA's last unit of an atom: reduce over the points, store, start afresh
#pragma unroll
            for (int lm = 0; lm < LM; ++lm)
                for (int off = L; off < 32; off <<= 1) acc[lm].add_shfl_xor(off);
            const int nrow = L < 32 ? NL_THREADS / 32 : rows;              // partial sums left per column
            const int row = L < 32 ? tid >> 5 : prow;
            const bool writer = L < 32 ? (tid & 31) < L : true;
            const size_t nout = (size_t)nlm * ncol;
#pragma unroll
            for (int l0 = 0; l0 < LM; l0 += NL_LMG) {      // NL_LMG lm values per pass through shared memory
                if (l0 >= nlm) break;
                __syncthreads();
                if (writer) {
#pragma unroll
                    for (int l = 0; l < NL_LMG; ++l)
                        if (l0 + l < LM) red[l][row * L + cl] = acc[l0 + l < LM ? l0 + l : 0];
                }
                __syncthreads();
                for (int e = tid; e < NL_LMG * L; e += NL_THREADS) {
                    const int l = e >> lshift, cc = e & (L - 1);
                    if (l0 + l >= nlm) continue;
                    V s = red[l][cc];
                    for (int r = 1; r < nrow; ++r) s.add(red[l][r * L + cc]);
                    s.st(partial + (size_t)d0.slot * nout + (size_t)(l0 + l) * ncol + cc * VEC);
                }
            }
#pragma unroll
            for (int lm = 0; lm < LM; ++lm) acc[lm] = V{};
        }
        d0 = d1, d1 = d2, d2 = d3, d3 = next(d3);
    }
    cp_async_wait<0>();
}

// P[atom][lm][c] = h3 * sum of the atom's partial sums, slots ascending: one CTA per atom that has sphere points
template <int VEC>
__global__ void __launch_bounds__(128) nl_finalize_kernel(const int4 *__restrict__ atom_slots, int nout, double h3,
                                                         const double *__restrict__ partial, double *__restrict__ P)
{
    using V = nl_vec<VEC>;
    pdl_launch_dependents();
    const int4 as = atom_slots[blockIdx.x];               // (atom, first slot, slots, -)
    pdl_wait();                                            // the partials of part 1
    for (int e = threadIdx.x * VEC; e < nout; e += 128 * VEC) {
        V s{};
        for (int k0 = 0; k0 < as.z; k0 += 4) {             // four loads in flight, added in slot order
            V t[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) t[j] = k0 + j < as.z ? V::ld(partial + (size_t)(as.y + k0 + j) * nout + e) : V{};
#pragma unroll
            for (int j = 0; j < 4; ++j) s.add(t[j]);
        }
        s.scale(h3);
        s.st(P + (size_t)as.x * nout + e);
    }
}

// Part 2: hpsi[u.ip][c] += sum over the pairs (q, A) that cover point u of sum_lm gamma[q][lm] P[A][lm][c].
// urec[u] = (mesh point, q of the first pair, its atom | (further pairs << 24), where the further pairs start in uext):
// nearly every point lies in one sphere, so one 16-byte record starts all of a point's loads at once.
template <int VEC, int LM>
__global__ void __launch_bounds__(NL_THREADS, NL_GATHER_CPS) nl_gather_kernel(int nu, const int4 *__restrict__ urec, const int2 *__restrict__ uext,
                                                              const double *__restrict__ gamma, int nlm, const double *__restrict__ P,
                                                              double *__restrict__ hpsi, int ncol, int lshift)
{
    using V = nl_vec<VEC>;
    const int tid = threadIdx.x, L = 1 << lshift, cl = tid & (L - 1), rows = NL_THREADS >> lshift;
    const int c = cl * VEC;
    const int per = rows * NL_GPT, nbatch = (nu + per - 1) / per;
    auto load_rec = [&](int batch, int4 (&r)[NL_GPT]) {
        const int u0 = batch * per + (tid >> lshift);
#pragma unroll
        for (int k = 0; k < NL_GPT; ++k) r[k] = batch < nbatch && u0 + k * rows < nu ? urec[u0 + k * rows] : make_int4(-1, 0, 0, 0);
    };
    // persistent CTAs over batches of rows * NL_GPT points; the records of the next batch are loaded while the Hpsi rows
    // of this one are in flight, so a batch costs one trip to memory, not two
    int4 rec[NL_GPT], nxt[NL_GPT];
    load_rec(blockIdx.x, rec);
    bool waited = false;
    for (int batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
        V h[NL_GPT];
#pragma unroll
        for (int k = 0; k < NL_GPT; ++k) h[k] = rec[k].x >= 0 ? V::ld(hpsi + (size_t)rec[k].x * ncol + c) : V{};
        load_rec(batch + gridDim.x, nxt);
        if (!waited) pdl_wait(), waited = true;            // P of this call
#pragma unroll
        for (int k = 0; k < NL_GPT; ++k) {
            if (rec[k].x < 0) continue;
            const double *g = gamma + (size_t)rec[k].y * nlm;
            const double *p = P + (size_t)(rec[k].z & 0xffffff) * nlm * ncol + c;   // 4-10 KB per atom: L1-resident
            V s{};
#pragma unroll
            for (int lm = 0; lm < LM; ++lm)
                if (lm < nlm) s.fma_(g[lm], V::ld(p + (size_t)lm * ncol));
            for (int e = rec[k].w, ee = e + (rec[k].z >> 24); e < ee; ++e) {
                const int2 qa = uext[e];
                g = gamma + (size_t)qa.x * nlm;
                p = P + (size_t)qa.y * nlm * ncol + c;
                for (int lm = 0; lm < nlm; ++lm) s.fma_(g[lm], V::ld(p + (size_t)lm * ncol));
            }
            h[k].add(s);
            h[k].st(hpsi + (size_t)rec[k].x * ncol + c);
        }
#pragma unroll
        for (int k = 0; k < NL_GPT; ++k) rec[k] = nxt[k];
    }
    if (!waited) pdl_wait();
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
    cudaFree(nl->d_idx), cudaFree(nl->d_gamma), cudaFree(nl->d_partial), cudaFree(nl->d_items), cudaFree(nl->d_P);
    cudaFree(nl->d_urec), cudaFree(nl->d_uext), cudaFree(nl->d_atom_slots);
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
    // work items of part 1: chunks of NL_CHUNK sphere points, atom after atom
    for (int A = 0; A < natoms; ++A) {
        const int64_t n = nl->off[A + 1] - nl->off[A];
        const int nch = (int)((n + NL_CHUNK - 1) / NL_CHUNK);
        for (int k = 0; k < nch; ++k)
            nl->items.push_back({A, (int32_t)(nl->off[A] + (int64_t)k * NL_CHUNK), (int32_t)std::min<int64_t>(NL_CHUNK, n - (int64_t)k * NL_CHUNK), -1});
    }
    // part 2: the union of the spheres, points ascending; per point the covering (sphere point, atom) pairs, atoms ascending
    {
        std::vector<int32_t> slot(m->np, -1);
        for (int A = 0; A < natoms; ++A)
            for (int64_t q = nl->off[A]; q < nl->off[A + 1]; ++q) slot[nl->idx[q]] = 0;
        for (int64_t ip = 0; ip < m->np; ++ip)
            if (slot[ip] == 0) {
                slot[ip] = (int32_t)nl->urec.size();
                nl->urec.push_back(make_int4((int)ip, -1, 0, 0));
            }
        std::vector<std::pair<int32_t, int2>> extra;
        for (int A = 0; A < natoms; ++A)
            for (int64_t q = nl->off[A]; q < nl->off[A + 1]; ++q) {
                int4 &r = nl->urec[slot[nl->idx[q]]];
                if (r.y < 0)
                    r.y = (int)q, r.z = A;
                else
                    extra.push_back({slot[nl->idx[q]], make_int2((int)q, A)});
            }
        std::stable_sort(extra.begin(), extra.end(), [](const std::pair<int32_t, int2> &a, const std::pair<int32_t, int2> &b) { return a.first < b.first; });
        bool too_many = natoms >= (1 << 24);
        for (size_t e = 0; e < extra.size(); ++e) {
            int4 &r = nl->urec[extra[e].first];
            if ((r.z >> 24) == 0) r.w = (int)e;
            if ((r.z >> 24) >= 127) too_many = true;
            else r.z += 1 << 24;
            nl->uext.push_back(extra[e].second);
        }
        if (too_many) {
            delete nl;
            return rs_fail(RS_ERR_UNSUPPORTED, "rs_nonlocal_create: too many atoms, or more than 128 spheres over one point");
        }
    }
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
        // part 1 runs on persistent CTAs, CTA b taking the items [b n / G, (b + 1) n / G): consecutive items are mostly of
        // one atom, and a CTA reduces and stores a partial sum only where the atom changes or its range ends
        const int nitems = (int)nl->items.size();
        nl->nctas = std::max(1, std::min(nitems, (nl->m->sm_count > 0 ? nl->m->sm_count : 148) * nl_cps(nl->nlm)));
        nl->nslots = 0;
        nl->atom_slots.clear();
        for (int b = 0; b < nl->nctas; ++b) {
            const int i0 = (int)((long long)b * nitems / nl->nctas), i1 = (int)((long long)(b + 1) * nitems / nl->nctas);
            for (int i = i0; i < i1; ++i) {
                const bool flush = i == i1 - 1 || nl->items[i + 1].atom != nl->items[i].atom;
                nl->items[i].slot = flush ? nl->nslots : -1;
                if (!flush) continue;
                if (nl->atom_slots.empty() || nl->atom_slots.back().x != nl->items[i].atom)
                    nl->atom_slots.push_back(make_int4(nl->items[i].atom, nl->nslots, 0, 0));
                ++nl->atom_slots.back().z;
                ++nl->nslots;
            }
        }
#define NL_SMEM(VEC, LM) \
    RS_CUDA_TRY(cudaFuncSetAttribute(nl_project_kernel<VEC, LM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)nl_project_smem(VEC, LM, 0)))
        NL_SMEM(1, 4);
        NL_SMEM(1, 9);
        NL_SMEM(1, 16);
        NL_SMEM(2, 4);
        NL_SMEM(2, 9);
        NL_SMEM(2, 16);
#undef NL_SMEM
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_idx, std::max<size_t>(16, nl->idx.size() * sizeof(int32_t))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_gamma, std::max<size_t>(16, nl->gamma.size() * sizeof(double))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_items, std::max<size_t>(16, nl->items.size() * sizeof(nl_item))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_partial, std::max<size_t>(16, (size_t)nl->nslots * nl->nlm * 128 * sizeof(double))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_P, (size_t)nl->natoms * nl->nlm * 128 * sizeof(double)));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_atom_slots, std::max<size_t>(16, nl->atom_slots.size() * sizeof(int4))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_urec, std::max<size_t>(16, nl->urec.size() * sizeof(int4))));
        RS_CUDA_TRY(cudaMalloc((void **)&nl->d_uext, std::max<size_t>(16, nl->uext.size() * sizeof(int2))));
        RS_CUDA_TRY(cudaMemcpy(nl->d_atom_slots, nl->atom_slots.data(), nl->atom_slots.size() * sizeof(int4), cudaMemcpyHostToDevice));
        RS_CUDA_TRY(cudaMemcpy(nl->d_idx, nl->idx.data(), nl->idx.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
        RS_CUDA_TRY(cudaMemcpy(nl->d_items, nl->items.data(), nl->items.size() * sizeof(nl_item), cudaMemcpyHostToDevice));
        RS_CUDA_TRY(cudaMemcpy(nl->d_urec, nl->urec.data(), nl->urec.size() * sizeof(int4), cudaMemcpyHostToDevice));
        RS_CUDA_TRY(cudaMemcpy(nl->d_uext, nl->uext.data(), nl->uext.size() * sizeof(int2), cudaMemcpyHostToDevice));
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
    if (((uintptr_t)psi | (uintptr_t)hpsi) & 15) return rs_fail(RS_ERR_INVALID_ARG, "rs_nonlocal_apply: blocks must be 16-byte aligned");
    rs_status rc = rs_nonlocal_prepare(nl);
    if (rc != RS_OK) return rc;
    if (nl->items.empty()) return RS_OK;
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);   // gamma is real: a complex block is 2 nst independent real columns
    cudaStream_t st = (cudaStream_t)stream;
    const double h3 = nl->m->h * nl->m->h * nl->m->h;
    const int vec = ncol >= 2 ? 2 : 1, lshift = ilog2n(ncol / vec);
    const int nu = (int)nl->urec.size(), per = (NL_THREADS >> lshift) * NL_GPT;
    const unsigned g2 = (unsigned)std::min((nu + per - 1) / per, (nl->m->sm_count > 0 ? nl->m->sm_count : 148) * NL_GATHER_CPS);
    cudaError_t e1, e2, e3;
    const int nout = nl->nlm * ncol, nitems = (int)nl->items.size();
    const unsigned g1 = (unsigned)nl->nctas;               // persistent
    const size_t smem1 = nl_project_smem(vec, nl->nlm, lshift);
#define NL_LAUNCH(VEC, LM)                                                                                                                \
    e1 = nl_launch(nl_project_kernel<VEC, LM>, g1, NL_THREADS, smem1, st, false, nl->d_items, nitems, nl->d_idx, nl->d_gamma, nl->nlm,       \
                   (const double *)psi, ncol, lshift, nl->d_partial);                                                                      \
    e2 = nl_launch(nl_finalize_kernel<VEC>, (unsigned)nl->atom_slots.size(), 128, 0, st, true, nl->d_atom_slots, nout, h3,      \
                   nl->d_partial, nl->d_P);                                                                                                \
    e3 = nl_launch(nl_gather_kernel<VEC, LM>, g2, NL_THREADS, 0, st, true, nu, nl->d_urec, nl->d_uext, nl->d_gamma, nl->nlm, nl->d_P,         \
                   (double *)hpsi, ncol, lshift)
    if (vec == 2) {
        if (nl->nlm <= 4) { NL_LAUNCH(2, 4); }
        else if (nl->nlm <= 9) { NL_LAUNCH(2, 9); }
        else { NL_LAUNCH(2, 16); }
    } else {
        if (nl->nlm <= 4) { NL_LAUNCH(1, 4); }
        else if (nl->nlm <= 9) { NL_LAUNCH(1, 9); }
        else { NL_LAUNCH(1, 16); }
    }
#undef NL_LAUNCH
    RS_CUDA_TRY(e1);
    RS_CUDA_TRY(e2);
    RS_CUDA_TRY(e3);
    return RS_OK;
}
