// Plane-sweep kernel: the fused stencil + local potential (step a5; eq. 2 :41)
// as a 2.5-D streaming kernel for sm_100a.
//
// What differs from the paper's kernel (one thread per (point, orbital), every star arm
// a separate load through a neighbour table) and why:
//   * A CTA owns a (TY x TZ)-point tile of the lattice's (y, z) plane and C of the block's columns and
//     marches along x.  Plane p of the tile (plus its y/z halos, no corners) is staged in shared
//     memory once (cp.async, zero-filled where the lattice point is outside the mesh = reading S3);
//     the x arm never touches memory again: every thread keeps, per output it owns, the last n centre
//     values and n partial sums in registers (2n-deep register window).
//   * A thread owns a Q x P patch of (y, z) points and VEC adjacent columns, so the y/z arm operands
//     it reads from shared memory are shared between its outputs: QP + 2n(Q + P) reads for QP outputs
//     instead of (4n + 1) QP.  On B200 the shared-memory pipe (128 B/clk/SM), not HBM, bounds a kernel
//     that reads all 6n + 1 operands per output.
//   * The neighbour table is the compact per-(tile, plane, row) record {first index, occupancy mask}
//     of rs_internal.h: ~1 byte per point instead of 24n.
// Requires RS_ORDER_LEX (in-domain points of a z-row consecutive in memory) and a non-periodic mesh;
// anything else is served by the gather kernel.
#include <algorithm>

#include "rs_internal.h"

// ---------------------------------------------------------------------------------------------
// host: tiles, work items, row records
// ---------------------------------------------------------------------------------------------
void rs_sweep_build_host(const rs_mesh *m, int n, int ty, int tz, int max_planes, std::vector<rs_sweep_item> &items,
                         std::vector<rs_rowinfo> &rows, int64_t *active_lanes)
{
    const int nx = m->dims[0], ny = m->dims[1], nz = m->dims[2];
    const int nrows = ty + 2 * n, w = tz + 2 * n;
    items.clear();
    rows.clear();
    int64_t lanes = 0;
    auto point = [&](int x, int y, int z) -> int32_t {
        if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) return -1;
        return m->dense2point[rs_dense_index(m, x, y, z)];
    };
    for (int y0 = 0; y0 < ny; y0 += ty)
        for (int z0 = 0; z0 < nz; z0 += tz) {
            int xlo = nx, xhi = -1;  // planes where the tile interior holds a mesh point
            for (int x = 0; x < nx; ++x) {
                bool any = false;
                for (int y = y0; y < std::min(y0 + ty, ny) && !any; ++y)
                    for (int z = z0; z < std::min(z0 + tz, nz) && !any; ++z) any = point(x, y, z) >= 0;
                if (any) {
                    xlo = std::min(xlo, x);
                    xhi = std::max(xhi, x);
                }
            }
            if (xhi < xlo) continue;
            const int len = xhi - xlo + 1;
            const int nchunks = (len + max_planes - 1) / max_planes;
            for (int c = 0; c < nchunks; ++c) {
                rs_sweep_item it;
                it.y0 = y0;
                it.z0 = z0;
                it.xa = xlo + (int)((int64_t)len * c / nchunks);
                it.xb = xlo + (int)((int64_t)len * (c + 1) / nchunks);
                it.tab = (int64_t)rows.size();
                for (int p = it.xa - n; p < it.xb + n; ++p)
                    for (int r = 0; r < nrows; ++r) {
                        rs_rowinfo ri = {0, 0, 0};
                        const int y = y0 - n + r;
                        const bool halo_row = r < n || r >= ty + n;
                        for (int zp = halo_row ? n : 0; zp < (halo_row ? n + tz : w); ++zp) {
                            const int32_t idx = point(p, y, z0 - n + zp);
                            if (idx < 0) continue;
                            if (!ri.mask) ri.off = idx;
                            ri.mask |= (uint64_t)1 << zp;
                        }
                        rows.push_back(ri);
                    }
                lanes += (int64_t)(it.xb - it.xa) * ty * tz;
                items.push_back(it);
            }
        }
    // items that start at the same plane run together: neighbouring tiles then read their common
    // halo rows at about the same time and find them in L2.
    std::stable_sort(items.begin(), items.end(),
                     [](const rs_sweep_item &a, const rs_sweep_item &b) { return a.xa < b.xa; });
    if (active_lanes) *active_lanes = lanes;
}

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------
template <int VEC>
struct vec;
template <>
struct vec<1> {
    double x;
    static __device__ __forceinline__ vec zero() { return {0.0}; }
    __device__ __forceinline__ void fma(double w, const vec &v) { x = ::fma(w, v.x, x); }
    static __device__ __forceinline__ vec mul(double w, const vec &v) { return {w * v.x}; }
};
template <>
struct __align__(16) vec<2> {
    double x, y;
    static __device__ __forceinline__ vec zero() { return {0.0, 0.0}; }
    __device__ __forceinline__ void fma(double w, const vec &v)
    {
        x = ::fma(w, v.x, x);
        y = ::fma(w, v.y, y);
    }
    static __device__ __forceinline__ vec mul(double w, const vec &v) { return {w * v.x, w * v.y}; }
};

template <int BYTES>
__device__ __forceinline__ void cp_async_zfill(void *smem_dst, const void *gsrc, bool valid)
{
    const unsigned dst = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int sz = valid ? BYTES : 0;
    if constexpr (BYTES == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(gsrc), "r"(sz) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(PENDING) : "memory");
}

template <int N_, int VEC_, int C_, int TY_, int TZ_, int Q_, int P_, int S_>
struct sweep_traits {
    static constexpr int N = N_, VEC = VEC_, C = C_, TY = TY_, TZ = TZ_, Q = Q_, P = P_, S = S_;
    static constexpr int ROWS = TY + 2 * N, W = TZ + 2 * N;
    static constexpr int CV = C / VEC;                 // column vectors per point
    static constexpr int GZ = TZ / P, GY = TY / Q;     // patches per tile row / column
    static constexpr int THREADS = CV * GZ * GY;
    static constexpr int WG = W / P;                   // z groups per de-interleaved sub-row
    static constexpr int PLANE_VECS = ROWS * W * CV;
    static constexpr int RING = 16;                    // row-record ring (steps t-N .. t+S live)
    static constexpr size_t SMEM = (size_t)S * PLANE_VECS * VEC * 8 + (size_t)RING * ROWS * sizeof(rs_rowinfo);
    static constexpr int LOAD_PTS_FULL = TY * W + 2 * N * TZ;
    static constexpr int LOAD_PTS_CORE = TY * TZ;
    static_assert(C % VEC == 0 && TZ % P == 0 && TY % Q == 0 && W % P == 0, "tile / patch mismatch");
    static_assert(W <= 64, "z window must fit one 64-bit occupancy mask");
    static_assert((CV & (CV - 1)) == 0, "CV must be a power of two");
    static_assert(N + S < RING, "row-record ring too short");
    static_assert(THREADS >= ROWS && THREADS <= 1024, "bad thread count");
};

// shared-memory position (in vec units) of (row r, window position zp, column vector cv): the z axis
// is de-interleaved by P so that the P-strided patches of adjacent lanes are adjacent in memory.
template <class T>
__device__ __forceinline__ int smem_pos(int r, int zp, int cv)
{
    return ((r * T::P + zp % T::P) * T::WG + zp / T::P) * T::CV + cv;
}

template <class T, bool CORE_ONLY>
__device__ __forceinline__ void load_plane(vec<T::VEC> *stage, const rs_rowinfo *ring_slot, const double *psi,
                                           int ncol, int col0, int tid)
{
    constexpr int NPTS = CORE_ONLY ? T::LOAD_PTS_CORE : T::LOAD_PTS_FULL;
    constexpr int NEL = NPTS * T::CV;
#pragma unroll
    for (int k = 0; k < (NEL + T::THREADS - 1) / T::THREADS; ++k) {
        const int e = tid + k * T::THREADS;
        if (e < NEL) {
            const int pt = e / T::CV, cv = e % T::CV;
            int r, zp;
            if (CORE_ONLY) {
                r = T::N + pt / T::TZ;
                zp = T::N + pt % T::TZ;
            } else if (pt < T::TY * T::W) {
                r = T::N + pt / T::W;
                zp = pt % T::W;
            } else {
                const int q = pt - T::TY * T::W, rr = q / T::TZ;
                r = rr < T::N ? rr : rr + T::TY;
                zp = T::N + q % T::TZ;
            }
            const rs_rowinfo ri = ring_slot[r];
            const bool in = (ri.mask >> zp) & 1;
            const int idx = ri.off + __popcll(ri.mask & (((uint64_t)1 << zp) - 1));
            const double *src = psi + ((int64_t)(in ? idx : 0) * ncol + col0 + cv * T::VEC);
            cp_async_zfill<T::VEC * 8>(stage + smem_pos<T>(r, zp, cv), src, in);
        }
    }
}

template <class T>
__global__ void __launch_bounds__(T::THREADS, 1)
sweep_kernel(const rs_sweep_item *__restrict__ items, const rs_rowinfo *__restrict__ rows,
             const double *__restrict__ vloc, const double *__restrict__ psi, double *__restrict__ hpsi, int ncol,
             int ngroups, const __grid_constant__ rs_weights w)
{
    constexpr int N = T::N, Q = T::Q, P = T::P, S = T::S, ROWS = T::ROWS;
    using V = vec<T::VEC>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *data = reinterpret_cast<V *>(smem_raw);
    rs_rowinfo *ring = reinterpret_cast<rs_rowinfo *>(smem_raw + (size_t)S * T::PLANE_VECS * sizeof(V));

    const int tid = threadIdx.x;
    const rs_sweep_item it = items[blockIdx.x / ngroups];
    const int col0 = (blockIdx.x % ngroups) * T::C;
    const int steps = (it.xb - it.xa) + 2 * N;     // step t handles lattice plane xa - N + t
    const rs_rowinfo *tab = rows + it.tab;

    const int cv = tid % T::CV, g = (tid / T::CV) % T::GZ, yq = tid / (T::CV * T::GZ);
    const int base = ((Q * yq * P) * T::WG + g) * T::CV + cv;   // window corner (row Q*yq, zp P*g) of this thread
    const int colv = col0 + cv * T::VEC;

    // prologue: row records of steps 0..S-1, then the data of steps 0..S-2
    for (int e = tid; e < S * ROWS; e += T::THREADS)
        if (e / ROWS < steps) ring[e] = tab[e];
    __syncthreads();
#pragma unroll
    for (int s = 0; s < S - 1; ++s) {
        if (s < steps) {
            if (s < N || s >= steps - N)   // warm-up / tail planes: centre values only, no halo
                load_plane<T, true>(data + s * T::PLANE_VECS, ring + s * ROWS, psi, ncol, col0, tid);
            else
                load_plane<T, false>(data + s * T::PLANE_VECS, ring + s * ROWS, psi, ncol, col0, tid);
        }
        cp_async_commit();
    }

    V in[N][Q][P], acc[N][Q][P];
#pragma unroll
    for (int k = 0; k < N; ++k)
#pragma unroll
        for (int j = 0; j < Q; ++j)
#pragma unroll
            for (int i = 0; i < P; ++i) in[k][j][i] = V::zero(), acc[k][j][i] = V::zero();

    int stage = 0;  // t % S
    for (int t0 = 0; t0 < steps; t0 += N) {
#pragma unroll
        for (int PH = 0; PH < N; ++PH) {
            const int t = t0 + PH;
            if (t < steps) {
                cp_async_wait<S - 2>();
                __syncthreads();
                // row record of step t+S (one per thread < ROWS), parked in registers until the end of the step
                int4 rnext = make_int4(0, 0, 0, 0);
                const bool fetch = tid < ROWS && t + S < steps;
                if (fetch) rnext = __ldg(reinterpret_cast<const int4 *>(tab + (int64_t)(t + S) * ROWS + tid));
                // data of step t+S-1 into the stage that step t-1 has just released
                {
                    const int tl = t + S - 1;
                    if (tl < steps) {
                        int sl = stage + S - 1;
                        sl = sl >= S ? sl - S : sl;
                        V *dst = data + sl * T::PLANE_VECS;
                        const rs_rowinfo *slot = ring + (tl & (T::RING - 1)) * ROWS;
                        if (tl < N || tl >= steps - N)
                            load_plane<T, true>(dst, slot, psi, ncol, col0, tid);
                        else
                            load_plane<T, false>(dst, slot, psi, ncol, col0, tid);
                    }
                    cp_async_commit();
                }
                const V *sp = data + stage * T::PLANE_VECS + base;
                const bool full = t >= N && t < steps - N;
                V ctr[Q][P];
                V a[Q][P];
                if (full) {
                    // potential at the thread's own points (latency hidden behind the arm sums)
                    double vv[Q][P];
                    const rs_rowinfo *slot = ring + (t & (T::RING - 1)) * ROWS;
#pragma unroll
                    for (int j = 0; j < Q; ++j) {
                        const rs_rowinfo ri = slot[N + Q * yq + j];
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            const int zp = N + P * g + i;
                            const bool inb = (ri.mask >> zp) & 1;
                            const int idx = ri.off + __popcll(ri.mask & (((uint64_t)1 << zp) - 1));
                            vv[j][i] = inb ? __ldg(vloc + idx) : 0.0;
                        }
                    }
                    // z arms (and the centre values) of the thread's Q rows
#pragma unroll
                    for (int j = 0; j < Q; ++j) {
                        V v[P + 2 * N];
#pragma unroll
                        for (int tt = 0; tt < P + 2 * N; ++tt)
                            v[tt] = sp[(((N + j) * P + tt % P) * T::WG + tt / P) * T::CV];
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            ctr[j][i] = v[N + i];
                            V s = V::mul(w.w[1], v[N + i + 1]);
                            s.fma(w.w[1], v[N + i - 1]);
#pragma unroll
                            for (int k = 2; k <= N; ++k) {
                                s.fma(w.w[k], v[N + i + k]);
                                s.fma(w.w[k], v[N + i - k]);
                            }
                            a[j][i] = s;
                        }
                    }
                    // y arms of the thread's P columns
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        V u[Q + 2 * N];
#pragma unroll
                        for (int tt = 0; tt < Q + 2 * N; ++tt) {
                            if (tt >= N && tt < N + Q)
                                u[tt] = ctr[tt - N][i];
                            else
                                u[tt] = sp[((tt * P + (N + i) % P) * T::WG + (N + i) / P) * T::CV];
                        }
#pragma unroll
                        for (int j = 0; j < Q; ++j)
#pragma unroll
                            for (int k = 1; k <= N; ++k) {
                                a[j][i].fma(w.w[k], u[N + j + k]);
                                a[j][i].fma(w.w[k], u[N + j - k]);
                            }
                    }
                    // backward half of the x arm, centre term with the potential
#pragma unroll
                    for (int j = 0; j < Q; ++j)
#pragma unroll
                        for (int i = 0; i < P; ++i) {
#pragma unroll
                            for (int k = 1; k <= N; ++k) a[j][i].fma(w.w[k], in[(PH - k + N) % N][j][i]);
                            a[j][i].fma(3.0 * w.w[0] + vv[j][i], ctr[j][i]);
                        }
                } else {
#pragma unroll
                    for (int j = 0; j < Q; ++j)
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            ctr[j][i] = sp[(((N + j) * P + (N + i) % P) * T::WG + (N + i) / P) * T::CV];
                            a[j][i] = V::zero();
                        }
                }
                if (t >= N) {
                    // forward half of the x arm: this plane's centre values feed the n pending outputs
#pragma unroll
                    for (int k = 1; k <= N; ++k)
#pragma unroll
                        for (int j = 0; j < Q; ++j)
#pragma unroll
                            for (int i = 0; i < P; ++i) acc[(PH - k + N) % N][j][i].fma(w.w[k], ctr[j][i]);
                    if (t >= 2 * N) {
                        // the output of step t-N is complete
                        const rs_rowinfo *slot = ring + ((t - N) & (T::RING - 1)) * ROWS;
#pragma unroll
                        for (int j = 0; j < Q; ++j) {
                            const rs_rowinfo ri = slot[N + Q * yq + j];
#pragma unroll
                            for (int i = 0; i < P; ++i) {
                                const int zp = N + P * g + i;
                                if ((ri.mask >> zp) & 1) {
                                    const int idx = ri.off + __popcll(ri.mask & (((uint64_t)1 << zp) - 1));
                                    *reinterpret_cast<V *>(hpsi + ((int64_t)idx * ncol + colv)) = acc[PH][j][i];
                                }
                            }
                        }
                    }
                }
#pragma unroll
                for (int j = 0; j < Q; ++j)
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        acc[PH][j][i] = a[j][i];
                        in[PH][j][i] = ctr[j][i];
                    }
                if (fetch) reinterpret_cast<int4 *>(ring)[((t + S) & (T::RING - 1)) * ROWS + tid] = rnext;
                stage = stage + 1 == S ? 0 : stage + 1;
            }
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// variants and dispatch
// ---------------------------------------------------------------------------------------------
static int g_max_planes = 48;   // x-chunk length of a work item (rs_set_tuning("sweep_planes", v))
void rs_sweep_set_max_planes(int v) { g_max_planes = v < 8 ? 8 : v; }

template <class T>
static rs_status launch_variant(const rs_mesh *cm, const rs_weights &w, const double *vloc, const double *psi,
                                double *hpsi, int ncol, cudaStream_t st)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);  // lazily filled cache inside the handle
    const auto key = std::make_tuple(T::N, T::TY, T::TZ);
    auto f = m->sweep.find(key);
    if (f == m->sweep.end()) {
        std::vector<rs_sweep_item> items;
        std::vector<rs_rowinfo> rows;
        rs_sweep_tables tb;
        tb.n = T::N, tb.ty = T::TY, tb.tz = T::TZ;
        rs_sweep_build_host(m, T::N, T::TY, T::TZ, g_max_planes, items, rows, &tb.active_lanes);
        tb.nitems = (int64_t)items.size();
        tb.nrecords = (int64_t)rows.size();
        RS_CUDA_TRY(cudaMalloc(&tb.d_items, items.size() * sizeof(rs_sweep_item)));
        RS_CUDA_TRY(cudaMalloc(&tb.d_rows, rows.size() * sizeof(rs_rowinfo)));
        RS_CUDA_TRY(cudaMemcpy(tb.d_items, items.data(), items.size() * sizeof(rs_sweep_item), cudaMemcpyHostToDevice));
        RS_CUDA_TRY(cudaMemcpy(tb.d_rows, rows.data(), rows.size() * sizeof(rs_rowinfo), cudaMemcpyHostToDevice));
        f = m->sweep.emplace(key, tb).first;
    }
    static bool attr_set = false;
    if (!attr_set) {
        RS_CUDA_TRY(cudaFuncSetAttribute(sweep_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM));
        attr_set = true;
    }
    const rs_sweep_tables &tb = f->second;
    const int ngroups = ncol / T::C;
    const unsigned grid = (unsigned)(tb.nitems * ngroups);
    sweep_kernel<T><<<grid, T::THREADS, T::SMEM, st>>>(tb.d_items, tb.d_rows, vloc, psi, hpsi, ncol, ngroups, w);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

//                 N  VEC C  TY  TZ  Q  P  S
// Thread counts are multiples of 128 (one register-file partition per scheduler): 256 threads leave
// each thread up to 255 registers for its 2n-deep window over a 2 x 2 x VEC patch.
using sw4_c8 = sweep_traits<4, 2, 8, 16, 16, 2, 2, 3>;
using sw4_c4 = sweep_traits<4, 2, 4, 16, 32, 2, 2, 3>;
using sw4_c2 = sweep_traits<4, 2, 2, 32, 32, 2, 2, 3>;
using sw4_c1 = sweep_traits<4, 1, 1, 32, 32, 2, 2, 3>;

bool rs_sweep_supported(const rs_mesh *m, int n, int ncol)
{
    return m->ordering == RS_ORDER_LEX && !m->periodic && n == 4 && ncol >= 1;
}

template <class T>
static int64_t variant_table_bytes(const rs_mesh *m, int ncol)
{
    auto f = m->sweep.find(std::make_tuple(T::N, T::TY, T::TZ));
    if (f == m->sweep.end()) {   // not built yet: build on the host only to count
        std::vector<rs_sweep_item> items;
        std::vector<rs_rowinfo> rows;
        rs_sweep_build_host(m, T::N, T::TY, T::TZ, g_max_planes, items, rows, nullptr);
        return (int64_t)(rows.size() * sizeof(rs_rowinfo) + items.size() * sizeof(rs_sweep_item)) * (ncol / T::C);
    }
    return (f->second.nrecords * (int64_t)sizeof(rs_rowinfo) + f->second.nitems * (int64_t)sizeof(rs_sweep_item)) *
           (ncol / T::C);
}

#define RS_SWEEP_DISPATCH(n, ncol, CALL)                      \
    do {                                                      \
        if ((n) == 4) {                                       \
            if ((ncol) >= 8) { CALL(sw4_c8); }                \
            else if ((ncol) == 4) { CALL(sw4_c4); }           \
            else if ((ncol) == 2) { CALL(sw4_c2); }           \
            else { CALL(sw4_c1); }                            \
        }                                                     \
    } while (0)

rs_status rs_launch_sweep(const rs_mesh *m, int n, const rs_weights &w, const double *vloc, const double *psi,
                          double *hpsi, int ncol, cudaStream_t st)
{
#define CALL(T) return launch_variant<T>(m, w, vloc, psi, hpsi, ncol, st)
    RS_SWEEP_DISPATCH(n, ncol, CALL);
#undef CALL
    return rs_fail(RS_ERR_UNSUPPORTED, "no plane-sweep variant for this order");
}

int64_t rs_sweep_table_bytes(const rs_mesh *m, int n, int ncol)
{
#define CALL(T) return variant_table_bytes<T>(m, ncol)
    RS_SWEEP_DISPATCH(n, ncol, CALL);
#undef CALL
    return 0;
}

const char *rs_sweep_variant_name(const rs_mesh *, int n, int ncol)
{
    if (n == 4) return ncol >= 8 ? "sweep[n4 c8 16x16 q2p2 s3]" : ncol == 4 ? "sweep[n4 c4 16x32 q2p2 s3]"
                     : ncol == 2 ? "sweep[n4 c2 32x32 q2p2 s3]" : "sweep[n4 c1 32x32 q2p2 s3]";
    return "none";
}

void rs_sweep_free(rs_mesh *m)
{
    for (auto &kv : m->sweep) {
        if (kv.second.d_items) cudaFree(kv.second.d_items);
        if (kv.second.d_rows) cudaFree(kv.second.d_rows);
    }
    m->sweep.clear();
}
