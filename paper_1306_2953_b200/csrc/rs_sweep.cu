// Plane-sweep kernel: the fused stencil + local potential (step a5; eq. 2 :41)
// as a 2.5-D streaming kernel written for sm_100a (TMA bulk copies, mbarriers, tensor memory).
//
// What differs from the paper's kernel (one thread per (point, orbital), every star arm
// a separate load through a neighbour table) and why -- see DESIGN.md "Kernels":
//   * A CTA owns a 16 x 16 tile of the lattice's (y, z) plane and 16 block columns, and marches along
//     x.  Plane p of the tile plus its y/z halos (no corners) is staged in shared memory ONCE by
//     bulk async copies (cp.async.bulk, one per run of in-domain points of a z-row: such a run is
//     one contiguous span of the blocked array because the orbital index is fastest);
//     completion is tracked by an mbarrier per stage.  Lattice points outside the mesh are zero-filled
//     in shared memory (reading S3), so the compute code has no predicates.
//   * A thread owns a 4 x 4 patch of (y, z) points of ONE column (the 16 lanes of a half-warp are the
//     16 columns of a point: every shared-memory read is a conflict-free 128-byte row).  The y/z arm
//     operands are shared inside the patch: 5 shared-memory reads per output instead of 17.
//   * The x arm never touches shared memory: the forward half is accumulated into the 4 pending
//     outputs of each (y, z) column held in registers; the backward half needs the centre values of
//     the previous 4 planes, which are parked in TENSOR MEMORY (tcgen05.st / tcgen05.ld, 32x32b shape:
//     every thread owns one TMEM lane, i.e. a private 2 KB scratch with ~2.6x the bandwidth of shared
//     memory, measured).  No tensor-core arithmetic is involved: the path is not a contraction.
//   * The neighbour table is replaced by per-(tile, plane) records built once on the host: the list of
//     copy runs, zero-fill bits, the mesh index of each of the tile's 256 points (for V and for the
//     store) and a 2-bit mode per warp (empty / centre-only / full) that lets a warp skip the planes
//     in which its 4 x 8 region holds no mesh point.  The records expand to exactly the plain table of
//     rs_mesh_get_index_map (reading S15).
// Requires RS_ORDER_LEX (in-domain points of a z-row consecutive in memory), a non-periodic mesh,
// fd_order 4 and a block of 16 real columns (B = 16 real or B = 8 complex); anything else is served by
// the gather kernel.
#include <algorithm>

#include "rs_internal.h"

namespace {

constexpr int SW_N = 4;                  // half-width of the star
constexpr int SW_T = 16;                 // tile edge (points) in y and z
constexpr int SW_W = SW_T + 2 * SW_N;    // 24: rows / z-slots of a staged plane
constexpr int SW_C = 16;                 // columns per CTA
constexpr int SW_SLOT_BYTES = SW_C * 8;  // 128
constexpr int SW_STAGE_BYTES = SW_W * SW_W * SW_SLOT_BYTES;  // 73,728: uniform [24][24] slots, corners hold V and idx
constexpr int SW_STAGES = 3;
constexpr int SW_THREADS = 256;
constexpr int SW_MAXRUN = RS_SWEEP_MAXRUN;
constexpr int SW_TMEM_COLS = 512;        // allocated; used: 2 x (4 x 32 [centre ring] + 4 x 16 [index ring])
// packed per-plane record (rs_internal.h): runs | fill bits | header | indices of the tile's points
constexpr int SW_REC_RUNS = 0, SW_REC_FILL = SW_MAXRUN * 8, SW_REC_HDR = SW_REC_FILL + 64, SW_REC_CIDX = SW_REC_HDR + 16;
constexpr int SW_REC_BYTES = RS_SWEEP_REC_BYTES;
static_assert(SW_REC_BYTES == SW_REC_CIDX + 256 * 4 && SW_REC_BYTES % 16 == 0, "record layout");
constexpr int SW_RING = 4;               // record ring: record r is requested 3 steps before it is consumed
constexpr size_t SW_SMEM = (size_t)SW_STAGES * SW_STAGE_BYTES + (size_t)SW_RING * SW_REC_BYTES;

// ---------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.expect_tx.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// one contiguous span global -> shared, completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void cp_async8_zfill(uint32_t dst, const void *src, uint32_t src_bytes)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_arrive_noinc(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}

// ---- tensor memory: every thread reads / writes consecutive 32-bit columns of its own lane -------
#define R4(a, o) "r"(a[o]), "r"(a[o + 1]), "r"(a[o + 2]), "r"(a[o + 3])
#define W4(a, o) "=r"(a[o]), "=r"(a[o + 1]), "=r"(a[o + 2]), "=r"(a[o + 3])
#define P4(a, o) "+r"(a[o]), "+r"(a[o + 1]), "+r"(a[o + 2]), "+r"(a[o + 3])

__device__ __forceinline__ void tm_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
        : W4(r, 0), W4(r, 4), W4(r, 8), W4(r, 12)
        : "r"(taddr));
}
__device__ __forceinline__ void tm_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,"
        "%30,%31}, [%32];\n"
        : W4(r, 0), W4(r, 4), W4(r, 8), W4(r, 12), W4(r, 16), W4(r, 20), W4(r, 24), W4(r, 28)
        : "r"(taddr));
}
__device__ __forceinline__ void tm_st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n" ::"r"(taddr), R4(r, 0), R4(r, 4)
                 : "memory");
}
__device__ __forceinline__ void tm_st16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};\n" ::"r"(taddr),
        R4(r, 0), R4(r, 4), R4(r, 8), R4(r, 12)
        : "memory");
}
// The loaded registers are passed through the wait so that no use of them can be scheduled above it.
__device__ __forceinline__ void tm_wait_ld16(uint32_t (&r)[16])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" : P4(r, 0), P4(r, 4), P4(r, 8), P4(r, 12)::"memory");
}
__device__ __forceinline__ void tm_wait_ld32(uint32_t (&r)[32])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;\n"
                 : P4(r, 0), P4(r, 4), P4(r, 8), P4(r, 12), P4(r, 16), P4(r, 20), P4(r, 24), P4(r, 28)::"memory");
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }
#undef R4
#undef W4
#undef P4

__device__ __forceinline__ double words2double(uint32_t lo, uint32_t hi) { return __hiloint2double((int)hi, (int)lo); }

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
struct sweep_args {
    const int2 *items;           // {first record, number of steps}
    const unsigned char *recs;   // [nrec][SW_REC_BYTES] packed per-plane records
    const double *vloc;
    const double *psi;
    double *hpsi;
};

enum { MODE_EMPTY = 0, MODE_CENTRE = 1, MODE_FULL = 2 };
constexpr uint32_t HDR_OUTPUT_PLANE = 1u << 16;   // the plane has outputs: stage V and the indices

__global__ void __launch_bounds__(SW_THREADS, 1)
sweep_kernel(const __grid_constant__ sweep_args a, const __grid_constant__ rs_weights w)
{
    constexpr int N = SW_N;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint64_t full_bar[SW_STAGES];
    __shared__ uint64_t rec_bar[SW_RING];
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = tid & 15, patch = tid >> 4, py = patch >> 2, pz = patch & 3;
    const int2 item = a.items[blockIdx.x];
    const unsigned char *const recs = a.recs + (size_t)item.x * SW_REC_BYTES;
    const int nsteps = item.y;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < SW_STAGES; ++s) mbar_init(smem_u32(&full_bar[s]), SW_THREADS);
#pragma unroll
        for (int s = 0; s < SW_RING; ++s) mbar_init(smem_u32(&rec_bar[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&tmem_base_s)),
                     "n"(SW_TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    // this thread's TMEM lane (its warp's quarter) and the column range of its warp
    const uint32_t tbase = tmem_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(warp >> 2) * 192u;
    const uint32_t t_in = tbase;          // [patch row j][slot t mod 4][i]: centre values of the last 4 planes (doubles)
    const uint32_t t_ix = tbase + 128u;   // [slot t mod 4][16]: mesh indices of the last 4 planes' outputs

    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar0 = smem_u32(&full_bar[0]);
    const uint32_t rbar0 = smem_u32(&rec_bar[0]);
    unsigned char *const ring = smem + (size_t)SW_STAGES * SW_STAGE_BYTES;

    // ---- loader constants: two plane slots to zero-fill, one tile point for V and the index ----------
    uint32_t fill_off1, fill_off2;
    {
        const int e1 = tid, e2 = tid + 256;
        fill_off1 = (uint32_t)(((N + e1 / SW_W) * SW_W + e1 % SW_W) * SW_SLOT_BYTES);
        if (e2 < SW_T * SW_W)
            fill_off2 = (uint32_t)(((N + e2 / SW_W) * SW_W + e2 % SW_W) * SW_SLOT_BYTES);
        else {
            const int q = e2 - SW_T * SW_W, hr = q / SW_T;
            fill_off2 = (uint32_t)((((hr < N ? hr : hr + SW_T)) * SW_W + N + q % SW_T) * SW_SLOT_BYTES);
        }
    }
    const int ty = tid >> 4, tz = tid & 15;
    // corner A (rows 0..3, slots 0..3) holds V[16][16]; corner B (rows 0..3, slots 20..23) holds idx[16][16]
    const uint32_t v_off = (uint32_t)(((ty >> 2) * SW_W) * SW_SLOT_BYTES + ((ty & 3) * 16 + tz) * 8);
    const uint32_t i_off = (uint32_t)(((ty >> 2) * SW_W + SW_W - N) * SW_SLOT_BYTES + ((ty & 3) * 16 + tz) * 4);
    // ---- compute constants -------------------------------------------------------------------------
    const uint32_t b0 = (uint32_t)(((N + 4 * py) * SW_W + 4 * pz) * SW_SLOT_BYTES + c * 8);   // patch row 0, window slot 0
    const uint32_t vrow = (uint32_t)((py * SW_W) * SW_SLOT_BYTES + (4 * pz) * 8);
    const uint32_t irow = (uint32_t)((py * SW_W + SW_W - N) * SW_SLOT_BYTES + (4 * pz) * 4);

    // ---- record ring: record r lands in slot r mod 4, two steps before produce(r) reads it ----------------
    auto request_rec = [&](int r) {   // one thread
        const uint32_t bar = rbar0 + 8u * (r & (SW_RING - 1));
        fence_proxy_async();
        mbar_arrive_expect_tx(bar, SW_REC_BYTES);
        bulk_g2s(smem_u32(ring) + (uint32_t)(r & (SW_RING - 1)) * SW_REC_BYTES, recs + (size_t)r * SW_REC_BYTES, SW_REC_BYTES, bar);
    };
    // ---- producer: stage plane tl; returns the plane's header word ------------------------------------
    auto produce = [&](int tl, int stage_l) -> uint32_t {
        const int rs = tl & (SW_RING - 1);
        mbar_wait(rbar0 + 8u * rs, (uint32_t)(tl >> 2) & 1u);
        const unsigned char *rp = ring + (size_t)rs * SW_REC_BYTES;
        const uint32_t sb = sbase + (uint32_t)stage_l * SW_STAGE_BYTES;
        unsigned char *const sg = smem + (size_t)stage_l * SW_STAGE_BYTES;
        const uint32_t bar = bar0 + 8u * stage_l;
        if (warp == 0) {
            const uint2 r0 = *reinterpret_cast<const uint2 *>(rp + SW_REC_RUNS + lane * 8);
            const uint2 r1 = *reinterpret_cast<const uint2 *>(rp + SW_REC_RUNS + 256 + lane * 8);
            const uint32_t n0 = r0.y >> 16, n1 = r1.y >> 16;
            fence_proxy_async();
            if (n0 + n1) mbar_expect_tx(bar, (n0 + n1) * SW_SLOT_BYTES);
            if (n0) bulk_g2s(sb + (r0.y & 0xffffu) * SW_SLOT_BYTES, a.psi + (size_t)r0.x * SW_C, n0 * SW_SLOT_BYTES, bar);
            if (n1) bulk_g2s(sb + (r1.y & 0xffffu) * SW_SLOT_BYTES, a.psi + (size_t)r1.x * SW_C, n1 * SW_SLOT_BYTES, bar);
        }
        const uint32_t hdr = *reinterpret_cast<const uint32_t *>(rp + SW_REC_HDR);
        const uint32_t fb = *reinterpret_cast<const uint32_t *>(rp + SW_REC_FILL + (tid >> 4) * 4) >> (2 * (tid & 15));
        if (fb & 1u) {
            float4 *d = reinterpret_cast<float4 *>(sg + fill_off1);
#pragma unroll
            for (int q = 0; q < 8; ++q) d[q] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        if (fb & 2u) {
            float4 *d = reinterpret_cast<float4 *>(sg + fill_off2);
#pragma unroll
            for (int q = 0; q < 8; ++q) d[q] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        if (hdr & HDR_OUTPUT_PLANE) {
            const int32_t ci = *reinterpret_cast<const int32_t *>(rp + SW_REC_CIDX + tid * 4);
            *reinterpret_cast<int32_t *>(sg + i_off) = ci;
            if (ci >= 0) cp_async8_zfill(sb + v_off, a.vloc + ci, 8u);
        }
        cp_async_arrive_noinc(bar);
        return hdr;
    };

    if (tid == 0)
        for (int r = 0; r < SW_RING && r < nsteps; ++r) request_rec(r);
    uint32_t hdr_a = produce(0, 0);                 // nsteps >= 2 N + 1
    uint32_t hdr_b = produce(1, 1);

    double acc[N][4][4];   // pending outputs: acc[t mod 4] belongs to plane t
#pragma unroll
    for (int k = 0; k < N; ++k)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[k][j][i] = 0.0;

    int stage = 0;
    uint32_t parity = 0;
    const double w0x3 = 3.0 * w.w[0];
    double *const hp = a.hpsi + c;

    for (int t0 = 0; t0 < nsteps; t0 += N) {
#pragma unroll
        for (int PH = 0; PH < N; ++PH) {
            const int t = t0 + PH;
            if (t >= nsteps) break;
            // mesh indices of the outputs this step completes (plane t - 4); in flight during the barrier
            tm_wait_st();
            uint32_t io[16];
            tm_ld16(t_ix + PH * 16, io);
            mbar_wait(bar0 + 8u * stage, parity);
            __syncthreads();
            if (tid == 0 && t + SW_RING < nsteps) request_rec(t + SW_RING);
            uint32_t hdr_c = 0;
            if (t + SW_STAGES - 1 < nsteps) hdr_c = produce(t + SW_STAGES - 1, stage == 0 ? SW_STAGES - 1 : stage - 1);
            const int mode = (int)((hdr_a >> (2 * warp)) & 3u);
            const unsigned char *sp = smem + (size_t)stage * SW_STAGE_BYTES;
            const double *pb = reinterpret_cast<const double *>(sp + b0);

            uint32_t in_[16];   // this plane's output indices, parked for 4 steps
            if (mode == MODE_FULL) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int4 q = *reinterpret_cast<const int4 *>(sp + irow + j * 64);
                    in_[4 * j] = (uint32_t)q.x, in_[4 * j + 1] = (uint32_t)q.y, in_[4 * j + 2] = (uint32_t)q.z,
                            in_[4 * j + 3] = (uint32_t)q.w;
                }
            } else {
#pragma unroll
                for (int q = 0; q < 16; ++q) in_[q] = 0xffffffffu;
            }
            tm_wait_ld16(io);
            tm_st16(t_ix + PH * 16, in_);

            if (mode == MODE_FULL) {
                double ctr[4][4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint32_t pw[32];   // centre values of planes t-1 .. t-4 of this patch row
                    tm_ld32(t_in + j * 32, pw);
                    double v[4 + 2 * N];
#pragma unroll
                    for (int tt = 0; tt < 4 + 2 * N; ++tt) v[tt] = pb[(j * SW_W + tt) * SW_C];
                    const double2 va = *reinterpret_cast<const double2 *>(sp + vrow + j * 128);
                    const double2 vb = *reinterpret_cast<const double2 *>(sp + vrow + j * 128 + 16);
                    const double vv[4] = {va.x, va.y, vb.x, vb.y};
                    double s[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const double ce = v[N + i];
                        ctr[j][i] = ce;
#pragma unroll
                        for (int k = 1; k < N; ++k) acc[(PH + N - k) % N][j][i] = fma(w.w[k], ce, acc[(PH + N - k) % N][j][i]);
                        const double out = fma(w.w[N], ce, acc[PH][j][i]);
                        if ((int32_t)io[4 * j + i] >= 0) hp[(size_t)io[4 * j + i] * SW_C] = out;
                        s[i] = (w0x3 + vv[i]) * ce;
#pragma unroll
                        for (int k = 1; k <= N; ++k) {
                            s[i] = fma(w.w[k], v[N + i + k], s[i]);
                            s[i] = fma(w.w[k], v[N + i - k], s[i]);
                        }
                    }
                    // backward half of the x arm from tensor memory, then park this row's centre values
                    tm_wait_ld32(pw);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
#pragma unroll
                        for (int k = 1; k <= N; ++k) {
                            const int sl = (PH + N - k) % N;
                            s[i] = fma(w.w[k], words2double(pw[sl * 8 + 2 * i], pw[sl * 8 + 2 * i + 1]), s[i]);
                        }
                        acc[PH][j][i] = s[i];
                    }
                    uint32_t cw[8];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        cw[2 * i] = (uint32_t)__double2loint(ctr[j][i]);
                        cw[2 * i + 1] = (uint32_t)__double2hiint(ctr[j][i]);
                    }
                    tm_st8(t_in + j * 32 + PH * 8, cw);
                }
                // y arms: rows 4py-4 .. 4py+7 of the patch's 4 z columns
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    double u[4 + 2 * N];
#pragma unroll
                    for (int tt = 0; tt < 4 + 2 * N; ++tt)
                        u[tt] = (tt >= N && tt < N + 4) ? ctr[tt - N][i] : pb[((tt - N) * SW_W + N + i) * SW_C];
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int k = 1; k <= N; ++k) {
                            acc[PH][j][i] = fma(w.w[k], u[N + j + k], acc[PH][j][i]);
                            acc[PH][j][i] = fma(w.w[k], u[N + j - k], acc[PH][j][i]);
                        }
                }
            } else if (mode == MODE_CENTRE) {
                // centre-only plane (warm-up / tail of the work item): it feeds the x arms of its neighbours
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint32_t cw[8];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const double ce = pb[(j * SW_W + N + i) * SW_C];
#pragma unroll
                        for (int k = 1; k < N; ++k) acc[(PH + N - k) % N][j][i] = fma(w.w[k], ce, acc[(PH + N - k) % N][j][i]);
                        const double out = fma(w.w[N], ce, acc[PH][j][i]);
                        if ((int32_t)io[4 * j + i] >= 0) hp[(size_t)io[4 * j + i] * SW_C] = out;
                        acc[PH][j][i] = 0.0;
                        cw[2 * i] = (uint32_t)__double2loint(ce);
                        cw[2 * i + 1] = (uint32_t)__double2hiint(ce);
                    }
                    tm_st8(t_in + j * 32 + PH * 8, cw);
                }
            } else {
                // no mesh point of this warp's region in plane t: all centre values are zero
                uint32_t cw[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) cw[q] = 0u;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        if ((int32_t)io[4 * j + i] >= 0) hp[(size_t)io[4 * j + i] * SW_C] = acc[PH][j][i];
                        acc[PH][j][i] = 0.0;
                    }
                    tm_st8(t_in + j * 32 + PH * 8, cw);
                }
            }

            hdr_a = hdr_b;
            hdr_b = hdr_c;
            if (++stage == SW_STAGES) {
                stage = 0;
                parity ^= 1u;
            }
        }
    }
    tm_wait_st();
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base_s), "n"(SW_TMEM_COLS) : "memory");
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host: work items and per-plane records
// ---------------------------------------------------------------------------------------------
static int g_max_planes = 32;   // x-slab thickness of a work item (rs_set_tuning("sweep_planes", v))
void rs_sweep_set_max_planes(int v) { g_max_planes = v < 4 ? 4 : v; }

bool rs_sweep_build_host(const rs_mesh *m, int n, int max_planes, rs_sweep_host &out)
{
    if (n != SW_N) return false;
    const int N = SW_N, T = SW_T, W = SW_W;
    const int nx = m->dims[0], ny = m->dims[1], nz = m->dims[2];
    out = rs_sweep_host();
    auto point = [&](int x, int y, int z) -> int32_t {
        if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) return -1;
        return m->dense2point[rs_dense_index(m, x, y, z)];
    };
    // planes of each tile that hold a mesh point
    const int nty = (ny + T - 1) / T, ntz = (nz + T - 1) / T;
    std::vector<uint8_t> has((size_t)nty * ntz * nx, 0);
    for (int x = 0; x < nx; ++x)
        for (int y = 0; y < ny; ++y)
            for (int z = 0; z < nz; ++z)
                if (m->dense2point[rs_dense_index(m, x, y, z)] >= 0) has[((size_t)(y / T) * ntz + z / T) * nx + x] = 1;

    enum { UNKNOWN = 0, ZERO = 1, DATA = 2 };
    std::vector<uint8_t> state((size_t)SW_STAGES * W * W);
    for (int xs = 0; xs < nx; xs += max_planes) {            // slab-major: tiles of one slab run together and
        const int xe = std::min(nx, xs + max_planes);        // find their common halo rows in L2
        for (int iy = 0; iy < nty; ++iy)
            for (int iz = 0; iz < ntz; ++iz) {
                const uint8_t *h = &has[((size_t)iy * ntz + iz) * nx];
                int xa = -1, xb = -1;
                for (int x = xs; x < xe; ++x)
                    if (h[x]) {
                        if (xa < 0) xa = x;
                        xb = x + 1;
                    }
                if (xa < 0) continue;
                const int y0 = iy * T, z0 = iz * T;
                const int nsteps = (xb - xa) + 2 * N;
                out.items.push_back(make_int2((int)out.nrec, nsteps));
                std::fill(state.begin(), state.end(), (uint8_t)UNKNOWN);   // shared memory of a starting CTA is arbitrary
                for (int s = 0; s < nsteps; ++s) {
                    const int p = xa - N + s;
                    const bool full = s >= N && s < nsteps - N;
                    out.recs.resize((size_t)(out.nrec + 1) * SW_REC_BYTES, 0);
                    unsigned char *rec = out.recs.data() + (size_t)out.nrec * SW_REC_BYTES;
                    uint2 *runs = reinterpret_cast<uint2 *>(rec + SW_REC_RUNS);
                    uint32_t *fill = reinterpret_cast<uint32_t *>(rec + SW_REC_FILL);
                    uint32_t *hdrp = reinterpret_cast<uint32_t *>(rec + SW_REC_HDR);
                    int32_t *cidx = reinterpret_cast<int32_t *>(rec + SW_REC_CIDX);
                    uint8_t *st = &state[(size_t)(s % SW_STAGES) * W * W];
                    // copy runs, and zero-fill bits for the slots this plane reads that are outside the mesh and
                    // do not already hold zeros from an earlier plane staged in the same buffer
                    int nrun = 0;
                    auto fill_bit = [&](int e) {   // e: plane slot in loader order (core rows with z halo, then y halo rows)
                        const int thr = e & 255, which = e >> 8;
                        fill[thr >> 4] |= 1u << (2 * (thr & 15) + which);
                    };
                    for (int r = full ? 0 : N; r < (full ? W : N + T); ++r) {
                        const bool halo_row = r < N || r >= N + T;
                        const int zlo = (halo_row || !full) ? N : 0, zhi = (halo_row || !full) ? N + T : W;
                        int run_start = -1;
                        for (int zp = zlo; zp <= zhi; ++zp) {
                            const int32_t idx = zp < zhi ? point(p, y0 - N + r, z0 - N + zp) : -1;
                            if (idx >= 0) {
                                if (run_start < 0) run_start = zp;
                                st[r * W + zp] = DATA;
                            } else {
                                if (run_start >= 0) {
                                    if (nrun >= SW_MAXRUN) return false;
                                    const int32_t first = point(p, y0 - N + r, z0 - N + run_start);
                                    runs[nrun++] = make_uint2((uint32_t)first,
                                                              (uint32_t)(r * W + run_start) | ((uint32_t)(zp - run_start) << 16));
                                    run_start = -1;
                                }
                                if (zp < zhi && st[r * W + zp] != ZERO) {
                                    fill_bit(halo_row ? T * W + (r < N ? r : r - T) * T + (zp - N) : (r - N) * W + zp);
                                    st[r * W + zp] = ZERO;
                                }
                            }
                        }
                    }
                    // warp modes and the mesh indices of the tile's own points
                    uint32_t hdr = full ? HDR_OUTPUT_PLANE : 0u;
                    for (int wq = 0; wq < 8; ++wq) {
                        bool any = false;
                        for (int y = 4 * (wq >> 1); y < 4 * (wq >> 1) + 4 && !any; ++y)
                            for (int z = 8 * (wq & 1); z < 8 * (wq & 1) + 8 && !any; ++z) any = point(p, y0 + y, z0 + z) >= 0;
                        if (any) hdr |= (uint32_t)(full ? MODE_FULL : MODE_CENTRE) << (2 * wq);
                    }
                    for (int y = 0; y < T; ++y)
                        for (int z = 0; z < T; ++z) cidx[y * T + z] = full ? point(p, y0 + y, z0 + z) : -1;
                    *hdrp = hdr;
                    ++out.nrec;
                }
            }
    }
    return true;
}

bool rs_sweep_supported(const rs_mesh *m, int n, int ncol)
{
    return m->ordering == RS_ORDER_LEX && !m->periodic && n == SW_N && ncol == SW_C;
}

static rs_status get_tables(rs_mesh *m, int n, const rs_sweep_tables **out)
{
    auto f = m->sweep.find(n);
    if (f == m->sweep.end()) {
        rs_sweep_host h;
        rs_sweep_tables tb;
        tb.ok = rs_sweep_build_host(m, n, g_max_planes, h);
        if (tb.ok) {
            tb.nitems = (int64_t)h.items.size();
            tb.nrec = h.nrec;
            auto up = [&](void **d, const void *src, size_t bytes) -> cudaError_t {
                cudaError_t e = cudaMalloc(d, bytes);
                if (e != cudaSuccess) return e;
                tb.bytes += (int64_t)bytes;
                return cudaMemcpy(*d, src, bytes, cudaMemcpyHostToDevice);
            };
            RS_CUDA_TRY(up((void **)&tb.d_items, h.items.data(), h.items.size() * sizeof(int2)));
            RS_CUDA_TRY(up((void **)&tb.d_recs, h.recs.data(), h.recs.size()));
            RS_CUDA_TRY(cudaFuncSetAttribute(sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SW_SMEM));
        }
        f = m->sweep.emplace(n, tb).first;
    }
    *out = &f->second;
    return RS_OK;
}

rs_status rs_launch_sweep(const rs_mesh *cm, int n, const rs_weights &w, const double *vloc, const double *psi,
                          double *hpsi, int ncol, cudaStream_t st)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);  // lazily filled cache inside the handle
    if (!rs_sweep_supported(m, n, ncol)) return rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep kernel cannot serve this call");
    const rs_sweep_tables *tb = nullptr;
    rs_status rc = get_tables(m, n, &tb);
    if (rc != RS_OK) return rc;
    if (!tb->ok) return rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep tables: a plane needs more copy runs than a record holds");
    sweep_args a;
    a.items = tb->d_items, a.recs = tb->d_recs;
    a.vloc = vloc, a.psi = psi, a.hpsi = hpsi;
    sweep_kernel<<<(unsigned)tb->nitems, SW_THREADS, SW_SMEM, st>>>(a, w);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

// true when the sweep kernel will really serve (mesh, n, ncol): supported and its tables could be built
bool rs_sweep_usable(const rs_mesh *cm, int n, int ncol)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    if (!rs_sweep_supported(m, n, ncol) || !m->have_device) return false;
    const rs_sweep_tables *tb = nullptr;
    return get_tables(m, n, &tb) == RS_OK && tb->ok;
}

int64_t rs_sweep_table_bytes(const rs_mesh *cm, int n, int ncol)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    if (!rs_sweep_supported(m, n, ncol)) return 0;
    auto f = m->sweep.find(n);
    if (f != m->sweep.end()) return f->second.bytes;
    rs_sweep_host h;   // no device (or not built yet): count on the host
    if (!rs_sweep_build_host(m, n, g_max_planes, h)) return 0;
    return (int64_t)(h.items.size() * sizeof(int2) + h.recs.size());
}

const char *rs_sweep_variant_name(const rs_mesh *, int, int) { return "sweep[n4 c16 16x16 q4p4 tma+tmem s3]"; }

void rs_sweep_free(rs_mesh *m)
{
    for (auto &kv : m->sweep) {
        rs_sweep_tables &t = kv.second;
        cudaFree(t.d_items), cudaFree(t.d_recs);
    }
    m->sweep.clear();
}
