// Layout transforms (a4, a6) and the general gather kernel (a5, per-point neighbour table).
#include "rs_internal.h"

// ---------------------------------------------------------------------------------------------
// pack / unpack: tiled transpose through shared memory (Fig. 4 :107).
// Reads of `states` are contiguous along the point index, writes of `block` are contiguous along
// (point, orbital); the smem tile is [B][tp+1] (padded: conflict-free).
// Tile = tp points x B orbitals with tp * B = 2048 elements (tp a power of two in 32..256): 8 independent
// loads in flight per thread, reads of 256-byte runs of one orbital, writes of whole 128-byte block rows.
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ T zero_of();
template <>
__device__ __forceinline__ double zero_of<double>()
{
    return 0.0;
}
template <>
__device__ __forceinline__ double2 zero_of<double2>()
{
    return make_double2(0.0, 0.0);
}

template <typename T>
__global__ void __launch_bounds__(256) pack_kernel(const T *__restrict__ states, int64_t ld, int ist0, int nst_in, int B,
                                                   int logB, int logTP, int64_t np, T *__restrict__ block)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *tile = reinterpret_cast<T *>(smem_raw);
    const int tp = 1 << logTP, total = B << logTP;
    const int64_t ip0 = (int64_t)blockIdx.x << logTP;
#pragma unroll 4
    for (int idx = threadIdx.x; idx < total; idx += 256) {
        const int j = idx >> logTP, p = idx & (tp - 1);
        T v = zero_of<T>();
        if (j < nst_in && ip0 + p < np) v = __ldg(states + (int64_t)(ist0 + j) * ld + ip0 + p);
        tile[j * (tp + 1) + p] = v;
    }
    __syncthreads();
#pragma unroll 4
    for (int idx = threadIdx.x; idx < total; idx += 256) {
        const int p = idx >> logB, j = idx & (B - 1);
        if (ip0 + p <= np) block[((ip0 + p) << logB) + j] = tile[j * (tp + 1) + p];  // row np: zero slot
    }
}

template <typename T>
__global__ void __launch_bounds__(256) unpack_kernel(const T *__restrict__ block, int B, int logB, int logTP, int nst_in,
                                                     int64_t np, T *__restrict__ states, int64_t ld, int ist0)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *tile = reinterpret_cast<T *>(smem_raw);
    const int tp = 1 << logTP, total = B << logTP;
    const int64_t ip0 = (int64_t)blockIdx.x << logTP;
#pragma unroll 4
    for (int idx = threadIdx.x; idx < total; idx += 256) {
        const int p = idx >> logB, j = idx & (B - 1);
        if (ip0 + p < np) tile[j * (tp + 1) + p] = __ldg(block + ((ip0 + p) << logB) + j);
    }
    __syncthreads();
#pragma unroll 4
    for (int idx = threadIdx.x; idx < total; idx += 256) {
        const int j = idx >> logTP, p = idx & (tp - 1);
        if (j < nst_in && ip0 + p < np) states[(int64_t)(ist0 + j) * ld + ip0 + p] = tile[j * (tp + 1) + p];
    }
}

static int ilog2(int v)
{
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

static int tile_log2(int B)   // points per tile: 2048 / B clamped to 32 .. 256
{
    int tp = 2048 / B;
    tp = tp < 32 ? 32 : tp > 256 ? 256 : tp;
    return ilog2(tp);
}

rs_status rs_launch_pack(const rs_mesh *m, const void *states, int64_t ld, int ist0, int nst_in, int B, void *block,
                         int lanes, cudaStream_t st)
{
    const int ltp = tile_log2(B), tp = 1 << ltp;
    const unsigned grid = (unsigned)((m->np + 1 + tp - 1) / tp);
    const size_t esz = lanes == 2 ? 16 : 8;
    const size_t smem = (size_t)B * (tp + 1) * esz;
    if (lanes == 2)
        pack_kernel<double2><<<grid, 256, smem, st>>>((const double2 *)states, ld, ist0, nst_in, B, ilog2(B), ltp, m->np,
                                                      (double2 *)block);
    else
        pack_kernel<double><<<grid, 256, smem, st>>>((const double *)states, ld, ist0, nst_in, B, ilog2(B), ltp, m->np,
                                                     (double *)block);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

rs_status rs_launch_unpack(const rs_mesh *m, const void *block, int B, int nst_in, void *states, int64_t ld, int ist0,
                           int lanes, cudaStream_t st)
{
    const int ltp = tile_log2(B), tp = 1 << ltp;
    const unsigned grid = (unsigned)((m->np + tp - 1) / tp);
    const size_t esz = lanes == 2 ? 16 : 8;
    const size_t smem = (size_t)B * (tp + 1) * esz;
    if (lanes == 2)
        unpack_kernel<double2><<<grid, 256, smem, st>>>((const double2 *)block, B, ilog2(B), ltp, nst_in, m->np,
                                                        (double2 *)states, ld, ist0);
    else
        unpack_kernel<double><<<grid, 256, smem, st>>>((const double *)block, B, ilog2(B), ltp, nst_in, m->np,
                                                       (double *)states, ld, ist0);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

// ---------------------------------------------------------------------------------------------
// General gather kernel.  One thread per (point, VEC adjacent columns); the tpp = ncol/VEC threads
// of a point are adjacent lanes, so every gathered row is one contiguous, vectorised read along the
// orbital axis ("for each point of the stencil we load several values, one per
// orbital in the block, that are contiguous in memory").  The point's table row (6n int32) is read
// as 16-byte (n even) or 8-byte vectors; all lanes of a point read the same addresses, which the
// load unit serves as one broadcast transaction.  Arms that leave the mesh read the zero slot.
// Works for any enumeration and for periodic boxes; it is the fallback of the brick kernel.
// ---------------------------------------------------------------------------------------------
template <int VEC>
struct vec_t;
template <>
struct vec_t<1> {
    using type = double;
    static __device__ __forceinline__ type ld(const double *p) { return __ldg(p); }
    static __device__ __forceinline__ void fma(type &a, double w, type v) { a = ::fma(w, v, a); }
    static __device__ __forceinline__ type mul(double w, type v) { return w * v; }
};
template <>
struct vec_t<2> {
    using type = double2;
    static __device__ __forceinline__ type ld(const double *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }
    static __device__ __forceinline__ void fma(type &a, double w, type v)
    {
        a.x = ::fma(w, v.x, a.x);
        a.y = ::fma(w, v.y, a.y);
    }
    static __device__ __forceinline__ type mul(double w, type v) { return make_double2(w * v.x, w * v.y); }
};

template <int N, int VEC>
__global__ void __launch_bounds__(256) gather_kernel(const int32_t *__restrict__ map, const double *__restrict__ vloc,
                                                     const double *__restrict__ psi, double *__restrict__ hpsi,
                                                     int64_t np, int tshift, int ncol, rs_weights w)
{
    using V = vec_t<VEC>;
    using T = typename V::type;
    const int64_t gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t ip = gtid >> tshift;
    if (ip >= np) return;
    const int col = (int)(gtid & ((1 << tshift) - 1)) * VEC;
    const double *base = psi + col;
    constexpr int NS = 6 * N;
    int32_t idx[NS];
    if constexpr (N % 2 == 0) {
        const int4 *row = reinterpret_cast<const int4 *>(map + ip * NS);
#pragma unroll
        for (int q = 0; q < NS / 4; ++q) {
            const int4 t = __ldg(row + q);
            idx[4 * q] = t.x, idx[4 * q + 1] = t.y, idx[4 * q + 2] = t.z, idx[4 * q + 3] = t.w;
        }
    } else {
        const int2 *row = reinterpret_cast<const int2 *>(map + ip * NS);
#pragma unroll
        for (int q = 0; q < NS / 2; ++q) {
            const int2 t = __ldg(row + q);
            idx[2 * q] = t.x, idx[2 * q + 1] = t.y;
        }
    }
    const T c = V::ld(base + ip * ncol);
    T acc = V::mul(3.0 * w.w[0] + __ldg(vloc + ip), c);
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const int k = (s % (2 * N)) / 2 + 1;
        V::fma(acc, w.w[k], V::ld(base + (int64_t)idx[s] * ncol));
    }
    *reinterpret_cast<T *>(hpsi + ip * ncol + col) = acc;
}

template <int N>
static rs_status launch_gather_n(const rs_mesh *m, const rs_weights &w, const int32_t *d_map, const double *vloc,
                                 const double *psi, double *hpsi, int ncol, cudaStream_t st)
{
    const int vec = ncol >= 2 ? 2 : 1;
    const int tpp = ncol / vec;
    const int tshift = ilog2(tpp);
    const int64_t nthreads = m->np * tpp;
    const unsigned grid = (unsigned)((nthreads + 255) / 256);
    if (vec == 2)
        gather_kernel<N, 2><<<grid, 256, 0, st>>>(d_map, vloc, psi, hpsi, m->np, tshift, ncol, w);
    else
        gather_kernel<N, 1><<<grid, 256, 0, st>>>(d_map, vloc, psi, hpsi, m->np, tshift, ncol, w);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

rs_status rs_launch_gather(const rs_mesh *m, int n, const rs_weights &w, const int32_t *d_map, const double *vloc,
                           const double *psi, double *hpsi, int ncol, cudaStream_t st)
{
    switch (n) {
        case 1: return launch_gather_n<1>(m, w, d_map, vloc, psi, hpsi, ncol, st);
        case 2: return launch_gather_n<2>(m, w, d_map, vloc, psi, hpsi, ncol, st);
        case 3: return launch_gather_n<3>(m, w, d_map, vloc, psi, hpsi, ncol, st);
        case 4: return launch_gather_n<4>(m, w, d_map, vloc, psi, hpsi, ncol, st);
        case 5: return launch_gather_n<5>(m, w, d_map, vloc, psi, hpsi, ncol, st);
        case 6: return launch_gather_n<6>(m, w, d_map, vloc, psi, hpsi, ncol, st);
        case 7: return launch_gather_n<7>(m, w, d_map, vloc, psi, hpsi, ncol, st);
        case 8: return launch_gather_n<8>(m, w, d_map, vloc, psi, hpsi, ncol, st);
    }
    return rs_fail(RS_ERR_UNSUPPORTED, "fd_order out of range");
}
