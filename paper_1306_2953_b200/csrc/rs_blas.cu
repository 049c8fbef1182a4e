// Block operations between orbitals (sec. VIII: "copies, linear
// combinations, and dot products ... implemented on the GPU using the block-of-orbitals approach"; RMM-DIIS works
// on residuals, sec. III).  All of them stream whole blocks once: bound by HBM.
//
// Reductions are deterministic: every CTA owns a fixed set of block rows and a fixed slot of per-CTA partial sums
// in a scratch array owned by the mesh; a second, tiny kernel adds the slots in CTA order.  No atomics.
#include "rs_internal.h"

namespace {

constexpr int RED_THREADS = 256;

__device__ __forceinline__ double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }

// per real column c of the block (ncol real columns, complex = adjacent (re, im) pairs):
//   q0 = sum a b, q1 = sum a a, q2 = sum (b - eps a)^2, q3 = sum (a_re b_im - a_im b_re)  [complex dot only, on the re column]
// VEC = 2: a thread owns two adjacent columns (one complex element); VEC = 1: ncol == 1.
template <int VEC, int NQ, bool CPLX_DOT>
__global__ void __launch_bounds__(RED_THREADS) block_reduce_kernel(const double *__restrict__ a, const double *__restrict__ b,
                                                                   const double *__restrict__ eps, int lanes, int64_t np, int ncol,
                                                                   int tshift, double *__restrict__ partial)
{
    __shared__ double red[RED_THREADS * VEC];
    const int tid = threadIdx.x, tpp = 1 << tshift;           // threads per point
    const int cv = tid & (tpp - 1), prow = tid >> tshift, rpc = RED_THREADS >> tshift;
    const int col = cv * VEC;
    double e[VEC] = {}, acc[NQ][VEC] = {};
    if (NQ > 2 && eps)
#pragma unroll
        for (int v = 0; v < VEC; ++v) e[v] = eps[(col + v) / lanes];
    const int64_t stride = (int64_t)gridDim.x * rpc;
    auto accumulate = [&](const double (&x)[VEC], const double (&y)[VEC]) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            acc[0][v] = fma(x[v], y[v], acc[0][v]);
            if constexpr (NQ > 1 && !CPLX_DOT) acc[1][v] = fma(x[v], x[v], acc[1][v]);
            if constexpr (NQ > 2) {
                const double r = fma(-e[v], x[v], y[v]);
                acc[2][v] = fma(r, r, acc[2][v]);
            }
        }
        if constexpr (CPLX_DOT && VEC == 2) acc[NQ - 1][1] += x[0] * y[1] - x[1] * y[0];   // Im conj(a) b in the im column's last slot
    };
    // RED_UNROLL rows per thread in flight (a read-only stream is bound by the bytes in flight, not by the arithmetic);
    // the rows are still added in ascending order
    constexpr int RED_UNROLL = 4;
    int64_t ip = (int64_t)blockIdx.x * rpc + prow;
    for (; ip + (RED_UNROLL - 1) * stride < np; ip += RED_UNROLL * stride) {
        double x[RED_UNROLL][VEC], y[RED_UNROLL][VEC];
#pragma unroll
        for (int u = 0; u < RED_UNROLL; ++u) {
            const int64_t o = (ip + u * stride) * ncol + col;
            if constexpr (VEC == 2) {
                const double2 xa = ld2(a + o), yb = ld2(b + o);
                x[u][0] = xa.x, x[u][1] = xa.y, y[u][0] = yb.x, y[u][1] = yb.y;
            } else {
                x[u][0] = a[o], y[u][0] = b[o];
            }
        }
#pragma unroll
        for (int u = 0; u < RED_UNROLL; ++u) accumulate(x[u], y[u]);
    }
    for (; ip < np; ip += stride) {
        double x[VEC], y[VEC];
        if constexpr (VEC == 2) {
            const double2 xa = ld2(a + ip * ncol + col), yb = ld2(b + ip * ncol + col);
            x[0] = xa.x, x[1] = xa.y, y[0] = yb.x, y[1] = yb.y;
        } else {
            x[0] = a[ip * ncol + col], y[0] = b[ip * ncol + col];
        }
        accumulate(x, y);
    }
    // CTA reduction over the rows, fixed order; slot layout partial[cta][q][ncol]
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        __syncthreads();
#pragma unroll
        for (int v = 0; v < VEC; ++v) red[tid * VEC + v] = acc[q][v];
        __syncthreads();
        if (prow == 0) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                double s = 0.0;
                for (int r = 0; r < rpc; ++r) s += red[((r << tshift) + cv) * VEC + v];
                partial[((size_t)blockIdx.x * NQ + q) * ncol + col + v] = s;
            }
        }
    }
}

// One warp per output: lane l adds the slots of CTAs l, l + 32, ... in that order, then a fixed butterfly adds the 32 lane
// sums: the same bits on every run.  mode 0: out[q][j] = sum over CTAs and over the orbital's lanes of partial[cta][q][j*lanes + l];
// mode 1 (complex dot, nq == 2): out[j] = (re, im), re = q0 over both lanes, im = the cross terms kept in the im column of q1.
__global__ void __launch_bounds__(256) block_reduce_final_kernel(const double *__restrict__ partial, int nctas, int nq, int nq_out,
                                                                 int ncol, int lanes, int mode, double *__restrict__ out)
{
    const int nst = ncol / lanes, lane = threadIdx.x & 31;
    const int idx = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (idx >= nq_out * nst) return;
    const int q = idx / nst, j = idx % nst;
    double s0 = 0.0, s1 = 0.0;
    // eight slots in flight per lane: all loads of a round are issued before the first add (a serial walk costs one
    // trip to L2 per slot: 37 trips = 25 us, measured), and the adds keep their order
    for (int c0 = lane; c0 < nctas; c0 += 32 * 8) {
        double t0[8], t1[8], t2[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int c = c0 + 32 * u;
            const bool in = c < nctas;
            const double *p0 = partial + ((size_t)(in ? c : 0) * nq + (mode == 1 ? 0 : q)) * ncol + (size_t)j * lanes;
            t0[u] = in ? p0[0] : 0.0;
            t1[u] = in && lanes == 2 ? p0[1] : 0.0;
            t2[u] = in && mode == 1 ? p0[ncol + 1] : 0.0;       // complex dot: the cross terms in the im column of q1
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (mode == 1) s0 += t0[u] + t1[u], s1 += t2[u];
            else if (lanes == 2) s0 += t0[u], s0 += t1[u];
            else s0 += t0[u];
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, o);
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    }
    if (lane == 0) {
        if (mode == 1)
            out[2 * j] = s0, out[2 * j + 1] = s1;
        else
            out[(size_t)q * nst + j] = s0;
    }
}

// y[p][c] += alpha_j x[p][c], rows p < np; complex: (yr, yi) += (ar xr - ai xi, ar xi + ai xr)
template <bool CPLX>
__global__ void __launch_bounds__(256) block_axpy_kernel(const double *__restrict__ alpha, const double *__restrict__ x,
                                                         double *__restrict__ y, int64_t nelem2, int ncol2)
{
    // one thread per pair of adjacent doubles (a complex element, or two real columns)
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nelem2; i += (int64_t)gridDim.x * blockDim.x) {
        const int c2 = (int)(i % ncol2);
        const double2 xv = ld2(x + 2 * i);
        double2 yv = ld2(y + 2 * i);
        if constexpr (CPLX) {
            const double ar = alpha[2 * c2], ai = alpha[2 * c2 + 1];
            yv.x += ar * xv.x - ai * xv.y;
            yv.y += ar * xv.y + ai * xv.x;
        } else {
            yv.x = fma(alpha[2 * c2], xv.x, yv.x);
            yv.y = fma(alpha[2 * c2 + 1], xv.y, yv.y);
        }
        *reinterpret_cast<double2 *>(y + 2 * i) = yv;
    }
}
__global__ void __launch_bounds__(256) block_axpy1_kernel(const double *__restrict__ alpha, const double *__restrict__ x,
                                                          double *__restrict__ y, int64_t np)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < np; i += (int64_t)gridDim.x * blockDim.x)
        y[i] = fma(alpha[0], x[i], y[i]);
}

int ilog2i(int v)
{
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

}  // namespace

// Scratch of per-CTA partial sums, owned by the mesh (allocated with it): RS_RED_CTAS x 4 quantities x 128 columns.
rs_status rs_reduce_scratch(const rs_mesh *cm, double **out)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    if (!m->d_red) RS_CUDA_TRY(cudaMalloc((void **)&m->d_red, (size_t)RS_RED_CTAS * 4 * 128 * sizeof(double)));
    *out = m->d_red;
    return RS_OK;
}

// mode 0: out[q][nst] for q < nq (1: <a|b> real part per orbital, 2: + |a|^2, 3: + |b - eps a|^2);  mode 1: complex dot (re, im)
rs_status rs_launch_block_reduce(const rs_mesh *m, const double *a, const double *b, const double *eps, int ncol, int lanes,
                                 int nq, int mode, double *out, cudaStream_t st)
{
    double *partial = nullptr;
    rs_status rc = rs_reduce_scratch(m, &partial);
    if (rc != RS_OK) return rc;
    const int vec = ncol >= 2 ? 2 : 1;
    const int tshift = ilog2i(ncol / vec);
    const int rpc = RED_THREADS >> tshift;
    int grid = (int)((m->np + rpc - 1) / rpc);
    const int cap = (m->sm_count > 0 ? m->sm_count : 148) * 8;
    if (grid > cap) grid = cap;
    if (grid > RS_RED_CTAS) grid = RS_RED_CTAS;
    const int nq_out = nq;    // rows of `out`; the partial sums may hold more quantities than asked for
    if (vec == 1)
        block_reduce_kernel<1, 3, false><<<grid, RED_THREADS, 0, st>>>(a, b, eps, lanes, m->np, ncol, tshift, partial), nq = 3;
    else if (mode == 1)
        block_reduce_kernel<2, 2, true><<<grid, RED_THREADS, 0, st>>>(a, b, nullptr, lanes, m->np, ncol, tshift, partial), nq = 2;
    else if (nq == 1)
        block_reduce_kernel<2, 1, false><<<grid, RED_THREADS, 0, st>>>(a, b, nullptr, lanes, m->np, ncol, tshift, partial);
    else
        block_reduce_kernel<2, 3, false><<<grid, RED_THREADS, 0, st>>>(a, b, eps, lanes, m->np, ncol, tshift, partial), nq = 3;
    RS_CUDA_TRY(cudaGetLastError());
    block_reduce_final_kernel<<<(nq_out * (ncol / lanes) * 32 + 255) / 256, 256, 0, st>>>(partial, grid, nq, nq_out, ncol, lanes, mode, out);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

rs_status rs_launch_block_axpy(const rs_mesh *m, const double *alpha, const double *x, double *y, int ncol, int lanes, cudaStream_t st)
{
    const int cap = (m->sm_count > 0 ? m->sm_count : 148) * 16;
    if (ncol == 1) {
        int grid = (int)((m->np + 255) / 256);
        block_axpy1_kernel<<<grid > cap ? cap : grid, 256, 0, st>>>(alpha, x, y, m->np);
    } else {
        const int64_t n2 = m->np * (int64_t)(ncol / 2);
        int grid = (int)((n2 + 255) / 256 > cap ? cap : (n2 + 255) / 256);
        if (lanes == 2)
            block_axpy_kernel<true><<<grid, 256, 0, st>>>(alpha, x, y, n2, ncol / 2);
        else
            block_axpy_kernel<false><<<grid, 256, 0, st>>>(alpha, x, y, n2, ncol / 2);
    }
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

// ---------------------------------------------------------------------------------------------
// rs_block_expectation_static: the expectation sums for callers that cannot allocate (code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc).  Same two kernels, same grid, same summation order as
// rs_block_expectation -- the results are bit-identical -- but the per-CTA partial sums go to a file-scope device
// array instead of the mesh-owned scratch that rs_reduce_scratch() allocates on first use.
//   * RS_STATIC_MAX_COLS real columns at most (nst <= 64 real, nst <= 32 complex): 1184 CTAs x 3 sums x 64 columns x
//     8 bytes = 1.73 MiB, which every GPU that loads the library holds until the process exits;
//   * nothing has to start at zero: every CTA of the first kernel overwrites all of its slots before the second
//     kernel reads them, so the previous call's contents do not matter;
//   * every call, on any mesh and any stream, shares the one array of its device: calls that overlap on the GPU race.
// In host code `rs_static_red` is a stand-in for the symbol, not a device address: its address is taken with
// cudaGetSymbolAddress, once per device, with that device current, and that pointer is what the kernels get.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr int RS_STATIC_MAX_COLS = 64;
constexpr int RS_STATIC_MAX_DEVICES = 64;
static __device__ __align__(256) double rs_static_red[(size_t)RS_RED_CTAS * 3 * RS_STATIC_MAX_COLS];

// address of rs_static_red on `device` (which must be current); resolved once per device, no allocation
rs_status static_red_address(int device, double **out)
{
    static double *addr[RS_STATIC_MAX_DEVICES] = {};
    if (device < 0 || device >= RS_STATIC_MAX_DEVICES) return rs_fail(RS_ERR_UNSUPPORTED, "rs_block_expectation_static: device ordinal");
    if (!addr[device]) {
        double *p = nullptr;
        RS_CUDA_TRY(cudaGetSymbolAddress((void **)&p, rs_static_red));
        if (!p) return rs_fail(RS_ERR_CUDA, "rs_block_expectation_static: cudaGetSymbolAddress returned a null address");
        addr[device] = p;   // racing first calls store the same value
    }
    *out = addr[device];
    return RS_OK;
}

}  // namespace

extern "C" rs_status rs_block_expectation_static(const rs_mesh *m, const void *psi, const void *hpsi, const double *eps_dev,
                                                 int nst, rs_dtype dtype, double *out_dev, void *stream)
{
    if (!m || !psi || !hpsi || !out_dev || nst < 1 || nst > RS_MAX_BLOCK || (nst & (nst - 1)) ||
        (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_block_expectation_static: bad argument");
    if ((((uintptr_t)psi | (uintptr_t)hpsi) & 15u) != 0)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_block_expectation_static: blocks must be 16-byte aligned");
    const int lanes = dtype == RS_COMPLEX128 ? 2 : 1, ncol = nst * lanes;
    if (ncol > RS_STATIC_MAX_COLS)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_block_expectation_static: " + std::to_string(ncol) + " real columns exceed the static scratch (" +
                                               std::to_string(RS_STATIC_MAX_COLS) + "): use rs_block_expectation");
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    int cur = -1;
    RS_CUDA_TRY(cudaGetDevice(&cur));
    if (cur != m->device) return rs_fail(RS_ERR_INVALID_ARG, "rs_block_expectation_static: the mesh's device must be current");
    double *partial = nullptr;
    rs_status rc = static_red_address(cur, &partial);
    if (rc != RS_OK) return rc;
    // the launch configuration of rs_launch_block_reduce(nq = 3, mode = 0), restated so that path stays as it is
    cudaStream_t st = (cudaStream_t)stream;
    const int vec = ncol >= 2 ? 2 : 1;
    const int tshift = ilog2i(ncol / vec);
    const int rpc = RED_THREADS >> tshift;
    int grid = (int)((m->np + rpc - 1) / rpc);
    const int cap = (m->sm_count > 0 ? m->sm_count : 148) * 8;
    if (grid > cap) grid = cap;
    if (grid > RS_RED_CTAS) grid = RS_RED_CTAS;
    const double *a = (const double *)psi, *b = (const double *)hpsi;
    if (vec == 1)
        block_reduce_kernel<1, 3, false><<<grid, RED_THREADS, 0, st>>>(a, b, eps_dev, lanes, m->np, ncol, tshift, partial);
    else
        block_reduce_kernel<2, 3, false><<<grid, RED_THREADS, 0, st>>>(a, b, eps_dev, lanes, m->np, ncol, tshift, partial);
    RS_CUDA_TRY(cudaGetLastError());
    block_reduce_final_kernel<<<(3 * nst * 32 + 255) / 256, 256, 0, st>>>(partial, grid, 3, 3, ncol, lanes, 0, out_dev);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}
