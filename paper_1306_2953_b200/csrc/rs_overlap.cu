// Overlap / subspace matrices over blocks of points:
//   M[j][k] = sum_p conj(a[p][j]) b[p][k]      S_jk = <phi_j|phi_k> (eq. 5, b = a)
//                                               h_jk = <phi_j|H|phi_k> (eq. 7, b = H phi)
// "we can use BLAS to calculate S as a rank k operation ... for a set of points at a time": the
// block layout [point][orbital] IS the paper's points-block array (all orbital coefficients of a point contiguous),
// so the contraction runs straight on the blocks: G = X^T Y over the real columns (a complex block = 2 real columns
// per orbital), accumulated over tiles of points.
//
// This is the one dense contraction on the path, so it runs on the fp64 tensor-core path: mma.sync m8n8k4 (DMMA),
// hand-written (no cuBLAS).  tcgen05 has no fp64 kind, so DMMA is what sm_100a offers for this arithmetic type.
//   * persistent CTAs (one to three per SM), each streaming its tiles of P points through a 3-stage cp.async ring;
//   * 8 warps: the (C/8)^2 output tiles of 8 x 8 are split into warp blocks of MT x NT tiles, the remaining
//     factor of 8 splits the points of a tile (K slices); row pitch padded to 4 (mod 16) doubles: the DMMA fragment
//     loads (lane -> point lane % 4, column lane / 4) are bank-conflict free;
//   * deterministic: per-CTA partial matrices go to a scratch array, a second kernel adds them in CTA order and
//     combines the real columns into complex entries.
#include "rs_internal.h"

namespace {

constexpr int OV_THREADS = 256;

template <int C_>
struct ov_shape {
    static constexpr int C = C_;                                        // real columns, padded to >= 8
    static constexpr int MT = C <= 8 ? 1 : C == 16 ? 2 : 4;             // 8 x 8 tiles per warp (rows)
    static constexpr int NT = C <= 8 ? 1 : C == 16 ? 2 : C <= 64 ? 4 : 8;
    static constexpr int WM = C / 8 / MT, WN = C / 8 / NT;              // warp blocks
    static constexpr int KS = 8 / (WM * WN);                            // K slices
    // points per stage / stages / CTAs per SM.  Blocks of <= 32 columns are bandwidth-bound and their tiles are small:
    // two or three CTAs per SM (independent barriers) keep more copies in flight than one CTA with a deeper ring
    // (measured, config 2: B = 16 0.120 -> 0.091 ms, B = 32 0.263 -> 0.185 ms); 64 columns: 32 x 32 warp blocks on two
    // CTAs per SM (0.73 -> 0.62 ms); 128 columns are bound by the DMMA rate.
    static constexpr int P = C <= 32 ? 64 : 32;
    static constexpr int STAGES = 3;
    static constexpr int CPS = C <= 16 ? 3 : C <= 64 ? 2 : 1;
    static constexpr int PITCH = C % 16 == 0 ? C + 4 : C == 8 ? 12 : 4; // doubles; = 4 or 12 (mod 16)
    static constexpr bool PAIRED = MT % 2 == 0 && NT % 2 == 0;   // 16-byte fragment loads (64 columns: 0.62 -> 0.56 ms)
    static constexpr int TILE = P * PITCH;                              // doubles per operand per stage
    static constexpr size_t SMEM_RING = (size_t)STAGES * 2 * TILE * 8;
    static constexpr size_t SMEM_RED = (size_t)KS * C * C * 8;
    static constexpr size_t SMEM = SMEM_RING > SMEM_RED ? SMEM_RING : SMEM_RED;
    static_assert(WM * WN * KS == 8 && P % (4 * KS) == 0 && SMEM <= 232448, "shape");
};

__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, int src_bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// x, y: blocks [np + 1][cr] (cr real columns, cr <= C; columns cr..C-1 of the shared tiles stay zero).  same = (x == y).
template <class S>
__global__ void __launch_bounds__(OV_THREADS, S::CPS) overlap_kernel(const double *__restrict__ x, const double *__restrict__ y, int64_t np,
                                                                int cr, int same, double *__restrict__ partial)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);
    constexpr int C = S::C, P = S::P, PITCH = S::PITCH, OV_STAGES = S::STAGES;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ks = warp % S::KS, wb = warp / S::KS, wm = wb / S::WN, wn = wb % S::WN;
    const int64_t ntiles = (np + P - 1) / P;

    // padding columns (cr < C) and the pitch padding are never written by the copies: clear the ring once
    for (int i = tid; i < OV_STAGES * 2 * S::TILE; i += OV_THREADS) ring[i] = 0.0;
    __syncthreads();

    const int chunks_row = cr / 2;                                    // 16-byte chunks per block row (cr >= 2)
    const int chunks = P * chunks_row;
    auto issue = [&](int64_t tile, int stage) {
        const int64_t p0 = tile * P;
        for (int op = 0; op < (same ? 1 : 2); ++op) {
            const double *src = (op ? y : x) + p0 * cr;
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(ring + ((size_t)stage * 2 + op) * S::TILE);
            for (int q = tid; q < chunks; q += OV_THREADS) {
                const int r = q / chunks_row, cc = q - r * chunks_row;
                const bool in = p0 + r < np;
                cp_async16(dst + (uint32_t)(r * PITCH + 2 * cc) * 8u, in ? (const void *)(src + (size_t)q * 2) : (const void *)x, in ? 16 : 0);
            }
        }
    };

    double acc[S::MT][S::NT][2] = {};
    int64_t tile = blockIdx.x;
    // prologue: OV_STAGES - 1 tiles in flight
    for (int s = 0; s < OV_STAGES - 1; ++s) {
        if (tile + (int64_t)s * gridDim.x < ntiles) issue(tile + (int64_t)s * gridDim.x, s);
        cp_async_commit();
    }
    int stage = 0;
    for (; tile < ntiles; tile += gridDim.x) {
        cp_async_wait<OV_STAGES - 2>();
        __syncthreads();   // this tile has landed for every thread; everyone is done with the stage refilled next
        {
            const int64_t nxt = tile + (int64_t)(OV_STAGES - 1) * gridDim.x;
            int ns = stage + OV_STAGES - 1;
            if (ns >= OV_STAGES) ns -= OV_STAGES;
            if (nxt < ntiles) issue(nxt, ns);
            cp_async_commit();
        }
        const double *xs = ring + (size_t)stage * 2 * S::TILE, *ys = same ? xs : xs + S::TILE;
        constexpr int KSTEPS = P / 4 / S::KS;
#pragma unroll 2
        for (int kk = 0; kk < KSTEPS; ++kk) {
            const int prow = (ks * KSTEPS + kk) * 4 + (lane & 3);
            double af[S::MT], bf[S::NT];
            if constexpr (S::PAIRED) {
                // one 16-byte load feeds two tiles: tile 2q takes the even, tile 2q + 1 the odd columns of a 16-column group
                // (the output indices below undo the interleave); quarter-warps stay bank-conflict free (pitch / 2 = 2 mod 8)
#pragma unroll
                for (int i = 0; i < S::MT; i += 2) {
                    const double2 t = *reinterpret_cast<const double2 *>(xs + prow * PITCH + (wm * S::MT + i) * 8 + 2 * (lane >> 2));
                    af[i] = t.x, af[i + 1] = t.y;
                }
#pragma unroll
                for (int j = 0; j < S::NT; j += 2) {
                    const double2 t = *reinterpret_cast<const double2 *>(ys + prow * PITCH + (wn * S::NT + j) * 8 + 2 * (lane >> 2));
                    bf[j] = t.x, bf[j + 1] = t.y;
                }
            } else {
#pragma unroll
                for (int i = 0; i < S::MT; ++i) af[i] = xs[prow * PITCH + (wm * S::MT + i) * 8 + (lane >> 2)];
#pragma unroll
                for (int j = 0; j < S::NT; ++j) bf[j] = ys[prow * PITCH + (wn * S::NT + j) * 8 + (lane >> 2)];
            }
#pragma unroll
            for (int i = 0; i < S::MT; ++i)
#pragma unroll
                for (int j = 0; j < S::NT; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
        if (++stage == OV_STAGES) stage = 0;
    }
    cp_async_wait<0>();
    __syncthreads();
    // K slices of the CTA -> one partial matrix, added in slice order
    double *red = reinterpret_cast<double *>(smem_raw);
#pragma unroll
    for (int i = 0; i < S::MT; ++i)
#pragma unroll
        for (int j = 0; j < S::NT; ++j) {
            int row = (wm * S::MT + i) * 8 + (lane >> 2), col = (wn * S::NT + j) * 8 + 2 * (lane & 3), col1 = col + 1;
            if constexpr (S::PAIRED) {
                row = (wm * S::MT + (i & ~1)) * 8 + 2 * (lane >> 2) + (i & 1);
                col = (wn * S::NT + (j & ~1)) * 8 + 4 * (lane & 3) + (j & 1);
                col1 = col + 2;
            }
            red[((size_t)ks * C + row) * C + col] = acc[i][j][0];
            red[((size_t)ks * C + row) * C + col1] = acc[i][j][1];
        }
    __syncthreads();
    for (int e = tid; e < C * C; e += OV_THREADS) {
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < S::KS; ++k) s += red[(size_t)k * C * C + e];
        partial[(size_t)blockIdx.x * C * C + e] = s;
    }
}

// M[j][k], j, k < nst: real: sum_cta G[j][k]; complex: (G[2j][2k] + G[2j+1][2k+1]) + i (G[2j][2k+1] - G[2j+1][2k]).
// One warp per entry: lane l adds the CTAs l, l + 32, ... in order, then a butterfly over the lanes: a fixed order
// (deterministic) without a serial walk over all CTAs.
__global__ void __launch_bounds__(256) overlap_final_kernel(const double *__restrict__ partial, int nctas, int C, int nst, int lanes,
                                                           double *__restrict__ M)
{
    const int lane = threadIdx.x & 31;
    const int idx = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (idx >= nst * nst) return;
    const int j = idx / nst, k = idx % nst;
    double re = 0.0, im = 0.0;
    if (lanes == 1) {
        for (int c = lane; c < nctas; c += 32) re += partial[(size_t)c * C * C + j * C + k];
    } else {
        for (int c = lane; c < nctas; c += 32) {
            const double *G = partial + (size_t)c * C * C;
            re += G[(2 * j) * C + 2 * k] + G[(2 * j + 1) * C + 2 * k + 1];
            im += G[(2 * j) * C + 2 * k + 1] - G[(2 * j + 1) * C + 2 * k];
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        re += __shfl_xor_sync(0xffffffffu, re, off);
        im += __shfl_xor_sync(0xffffffffu, im, off);
    }
    if (lane == 0) {
        if (lanes == 1) M[idx] = re;
        else M[2 * idx] = re, M[2 * idx + 1] = im;
    }
}

template <class S>
rs_status launch(const rs_mesh *m, const double *x, const double *y, int cr, double *partial, int grid, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        RS_CUDA_TRY(cudaFuncSetAttribute(overlap_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::SMEM));
        attr_set = true;
    }
    overlap_kernel<S><<<grid * S::CPS, OV_THREADS, S::SMEM, st>>>(x, y, m->np, cr, x == y ? 1 : 0, partial);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

}  // namespace

rs_status rs_overlap_scratch(const rs_mesh *cm, double **out)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    const int nctas = m->sm_count > 0 ? m->sm_count : 148;
    if (!m->d_ovl) RS_CUDA_TRY(cudaMalloc((void **)&m->d_ovl, (size_t)nctas * 128 * 128 * sizeof(double)));
    *out = m->d_ovl;
    return RS_OK;
}

// cr = real columns of both blocks (2 .. 128, a power of two); lanes 1 / 2; M_dev [nst][nst] elements
rs_status rs_launch_overlap(const rs_mesh *m, const double *x, const double *y, int cr, int lanes, double *M, cudaStream_t st)
{
    double *partial = nullptr;
    rs_status rc = rs_overlap_scratch(m, &partial);
    if (rc != RS_OK) return rc;
    const int nctas = m->sm_count > 0 ? m->sm_count : 148;
    const int C = cr < 8 ? 8 : cr;
    int cps = 1;
    switch (C) {
        case 8: rc = launch<ov_shape<8>>(m, x, y, cr, partial, nctas, st), cps = ov_shape<8>::CPS; break;
        case 16: rc = launch<ov_shape<16>>(m, x, y, cr, partial, nctas, st), cps = ov_shape<16>::CPS; break;
        case 32: rc = launch<ov_shape<32>>(m, x, y, cr, partial, nctas, st), cps = ov_shape<32>::CPS; break;
        case 64: rc = launch<ov_shape<64>>(m, x, y, cr, partial, nctas, st), cps = ov_shape<64>::CPS; break;
        case 128: rc = launch<ov_shape<128>>(m, x, y, cr, partial, nctas, st), cps = ov_shape<128>::CPS; break;
        default: return rs_fail(RS_ERR_INVALID_ARG, "rs_block_overlap: block width");
    }
    if (rc != RS_OK) return rc;
    overlap_final_kernel<<<(cr / lanes * (cr / lanes) + 7) / 8, 256, 0, st>>>(partial, nctas * cps, C, cr / lanes, lanes, M);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}
