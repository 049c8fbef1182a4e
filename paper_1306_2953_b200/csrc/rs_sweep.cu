// Plane-sweep kernel: the fused stencil + local potential (step a5; eq. 2 :41)
// as a persistent, warp-specialised 2.5-D streaming kernel for sm_100a (TMA copies, mbarriers,
// tensor memory, setmaxnreg).
//
// What differs from the paper's kernel (one thread per (point, orbital), every star arm
// a separate load through a neighbour table) and why -- see DESIGN.md "Kernels":
//   * One CTA per SM, persistent.  The host cuts the mesh into work items (a 16 x 16 tile of the
//     lattice's (y, z) plane x a slab of x planes x 16 block columns), orders them slab by slab (so
//     that tiles sharing halo rows run at about the same time and find them in L2) and deals them
//     to the CTAs with a cost model, splitting items in x where needed so that all CTAs finish together.
//     A CTA marches through its items plane by plane.
//   * Producer warp: stages plane p of the tile plus its y/z halo strips (no corners) in shared
//     memory ONCE, by bulk async copies -- one per run of in-domain points of a z-row: such a run
//     is one contiguous span of the blocked array because the orbital index is fastest;
//     for blocks wider than 16 columns the CTA takes a 16-column slice and the same runs become 2-D
//     tensor-map copies.  Completion is tracked by an mbarrier per stage (3 stages).  Lattice points
//     outside the mesh are zero-filled in shared memory (reading S3), so the arithmetic has no
//     predicates.  The producer also gathers V and the mesh indices of the tile's 256 points.
//   * 8 consumer warps, no block-wide barrier: they wait on the stage's "full" mbarrier and release it
//     through an "empty" mbarrier, so warps drift by up to two planes and hide each other's stalls.
//     A thread owns a 4 x 4 patch of (y, z) points of ONE column (the 16 lanes of a half-warp are the
//     16 columns of a point: every shared-memory read is a conflict-free 128-byte row).  The y/z arm
//     operands are shared inside the patch: 5 shared-memory reads per output instead of 17.
//   * The x arm never touches shared memory: the forward half is accumulated into the 4 pending
//     outputs of each (y, z) column held in registers; the backward half needs the centre values of
//     the previous 4 planes, which are parked in TENSOR MEMORY (tcgen05.st / tcgen05.ld, 32x32b shape:
//     every thread owns one TMEM lane, a private scratch).  No tensor-core arithmetic is involved:
//     the path is not a contraction.
//   * The neighbour table is replaced by per-(item, plane) records built once on the host: the list of
//     copy runs, zero-fill bits, the mesh index of each of the tile's 256 points (for V and for the
//     store) and a 2-bit mode per warp (empty / centre-only / full) that lets a warp skip the planes
//     in which its 4 x 8 region holds no mesh point.  The records expand to exactly the plain table of
//     rs_mesh_get_index_map (reading S15; rs_sweep_selfcheck verifies this on the host).
// The kernel is a template over its shape (star half-width, tile height, patch height, producer groups):
// fd_order 4 runs 16 x 16 tiles with 4 x 4 patches, fd_order 6 runs 8 x 16 tiles with 2 x 4 patches (6 pending
// planes of a 4 x 4 patch do not fit the register file).  The text below describes the fd_order 4 shape.
// Requires RS_ORDER_LEX (in-domain points of a z-row consecutive in memory), a non-periodic mesh,
// fd_order 4 or 6 and a block of 16, 32, 64 or 128 real columns; anything else is served by the gather kernel.
#include <cuda.h>

#include <algorithm>
#include <cmath>
#include <cstring>

#include "rs_internal.h"

namespace {

constexpr int SW_TZ = 16;                // tile edge (points) in z: one copy run per z-row
constexpr int SW_PZ = 4;                 // patch width in z: 4 patches across the tile
constexpr int SW_C = 16;                 // columns per CTA
constexpr int SW_SLOT_BYTES = SW_C * 8;  // 128
constexpr int SW_STAGES = 3;
constexpr int SW_MAXRUN = RS_SWEEP_MAXRUN;
constexpr int SW_TMEM_COLS = 512;
// packed per-plane record (rs_internal.h): runs | fill bitmap | header | clear list | indices of the tile's points
constexpr int SW_MAXFILL = 64;             // slots a record can list for clearing; more (a piece's first planes): the whole stage is cleared
constexpr int SW_REC_RUNS = 0, SW_REC_FILL = SW_MAXRUN * 8, SW_REC_HDR = SW_REC_FILL + 80, SW_REC_FLIST = SW_REC_HDR + 16,
              SW_REC_CIDX = SW_REC_FLIST + SW_MAXFILL * 2;
constexpr uint32_t HDR_NFILL_SHIFT = 16, HDR_NFILL_WHOLE = 0xffu;   // header word 0, bits 16..23: entries of the clear list, 0xff = clear the whole stage first
constexpr int SW_RING = 6;               // record ring of the producers
constexpr int SW_LOOKAHEAD = 3;          // records are requested this many steps ahead (SW_RING >= SW_LOOKAHEAD + 3)
constexpr int SW_NBOX = 6;               // tensor-map box heights 1, 2, 4, 8, 16, 24 (a run of 25..28 points takes two boxes)

// Kernel shape: star half-width N, tile of TY x 16 (y, z) points, register patch of PY x 4 points per thread,
// NGROUPS producer groups of 4 warps.  Compiled shapes (rs_sweep_variant()):
//   <4, 16, 4, 2>  fd_order 4: 8 consumer warps, 16 outputs per thread, 4 pending planes in registers
//   <6,  8, 2, 2>  fd_order 6: 6 pending planes of a 4 x 4 patch do not fit the register file; 2 x 4 patches do
template <int N_, int TY_, int PY_, int NGROUPS_, int GW_ = 4>
struct sweep_shape {
    static constexpr int N = N_, TY = TY_, PY = PY_, NGROUPS = NGROUPS_, GW = GW_;   // GW: warps per producer group
    static constexpr int WY = TY + 2 * N, WZ = SW_TZ + 2 * N;            // rows / z-slots of a staged plane
    static constexpr int STAGE_BYTES = WY * WZ * SW_SLOT_BYTES;         // uniform [WY][WZ] slots; the corners hold V, offsets, header
    static constexpr int NPT = TY * SW_TZ;                              // tile points
    static constexpr int CONSUMERS = (TY / PY) * (SW_TZ / SW_PZ) * SW_C;   // one thread per (patch, column)
    static constexpr int NCW = CONSUMERS / 32;
    static constexpr int PRODUCERS = 32 * GW * NGROUPS;
    static constexpr int THREADS = PRODUCERS + CONSUMERS;
    static constexpr int REC_BYTES = SW_REC_CIDX + NPT * 4;
    static constexpr int ROW_WORDS = N * 2 * SW_PZ;                      // tensor memory: one patch row = N ring slots x 4 doubles
    static constexpr size_t SMEM = (size_t)SW_STAGES * STAGE_BYTES + (size_t)SW_RING * REC_BYTES;
    // corner B (rows 0.., slots WZ-N..): the store offsets (4 tile rows = 256 bytes per corner row), then the header
    static constexpr uint32_t HDR_OFF = (uint32_t)(WZ - N + 2) * SW_SLOT_BYTES;
    // registers: THREADS x LAUNCH_REGS at launch = PRODUCERS x PROD_REGS + CONSUMERS x CONS_REGS at most
    static constexpr int LAUNCH_REGS = (65536 / THREADS) & ~7;
    static constexpr int PROD_REGS = 32;
    static constexpr int CONS_REGS = (LAUNCH_REGS + (LAUNCH_REGS - PROD_REGS) * PRODUCERS / CONSUMERS) & ~7;
    static_assert(TY % PY == 0 && 4 % PY == 0 && CONSUMERS % 128 == 0 && N % NGROUPS == 0 && (GW == 4 || GW == 8), "shape");
    static_assert(TY <= 4 * N && N >= 4, "the corners must hold V (512 bytes per corner row) and the offsets");
    static_assert(REC_BYTES % 16 == 0 && SMEM + 256 <= 232448, "shared memory budget");
    static_assert((NCW + 3) / 4 * PY * ROW_WORDS <= SW_TMEM_COLS, "tensor memory budget");
    static_assert(WY * WZ <= 18 * 32, "zero-fill bitmap");
};
// two groups of 4 producer warps alternate steps (one group of 8 warps staging every step was measured 4 % slower:
// 0.127 against 0.122 ms on config 2, B = 16)
using shape_n4 = sweep_shape<4, 16, 4, 2, 4>;
using shape_n6 = sweep_shape<6, 8, 2, 2, 4>;

// the same numbers at run time, for the host-side builder
struct shape_rt {
    int N, TY, PY, WY, WZ, NPT, NCW, rec_bytes;
};
template <class S>
shape_rt shape_of()
{
    return shape_rt{S::N, S::TY, S::PY, S::WY, S::WZ, S::NPT, S::NCW, S::REC_BYTES};
}

enum { MODE_EMPTY = 0, MODE_CENTRE = 1, MODE_FULL = 2 };
constexpr uint32_t HDR_OUTPUT_PLANE = 1u << 31;   // the plane has outputs: stage V and the indices (bits 0..23: 2 per warp)

// ---------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
// wait for the phase of `parity` to complete; the hardware suspends the warp (up to the hinted time) instead of spinning
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, %2;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity), "r"(100000u)
        : "memory");
}
// one contiguous span global -> shared, completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
// 2-D tensor-map copy: box {16 columns, box rows} at (column c0, row c1) -> shared, rows packed 128 B apart
__device__ __forceinline__ void tensor_g2s(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
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
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n" ::"r"(taddr), R4(r, 0), R4(r, 4));
}
// The loaded registers are passed through the wait so that no use of them can be scheduled above it.
__device__ __forceinline__ void tm_wait_ld16(uint32_t (&r)[16])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" : P4(r, 0), P4(r, 4), P4(r, 8), P4(r, 12));
}
__device__ __forceinline__ void tm_wait_ld32(uint32_t (&r)[32])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;\n"
                 : P4(r, 0), P4(r, 4), P4(r, 8), P4(r, 12), P4(r, 16), P4(r, 20), P4(r, 24), P4(r, 28));
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n"); }
#undef R4
#undef W4
#undef P4

// predicated 8-byte store to base + 8 * off unless off is the invalid mark: no branch, one address instruction
__device__ __forceinline__ void store_if_valid(double *base, uint32_t off, double v)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        ".reg .u64 q;\n"
        "setp.ne.u32 p, %0, 0xffffffff;\n"
        "mad.wide.u32 q, %0, 8, %1;\n"
        "@p st.global.cs.f64 [q], %2;\n"
        "}\n" ::"r"(off),
        "l"(base), "d"(v));   // no "memory" clobber: the compiler may move shared-memory loads across these stores
}

__device__ __forceinline__ double words2double(uint32_t lo, uint32_t hi) { return __hiloint2double((int)hi, (int)lo); }

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
struct sweep_args {
    const int2 *items;           // per CTA: {first record, number of steps}
    const unsigned char *recs;   // [nrec][REC_BYTES] packed per-plane records
    const double *vloc;
    const double *psi;
    double *hpsi;
    uint32_t ncol;               // row pitch of the block in elements
    long long *cycles;           // optional [gridDim.x]: clock64 ticks each CTA spent (calibration of the cost model)
    long long *step_clock;       // optional [nrec]: clock64 at the end of every step (rs_hamiltonian_autotune)
};
struct sweep_maps {
    CUtensorMap box[SW_NBOX];    // psi as a [np+1][ncol] fp64 tensor, box {16, 1|2|4|8|16|24}
};

// ---- producer warps: NGROUPS groups of 4 warps stage plane after plane, group g taking steps t = g (mod NGROUPS) ----
// Inside a group every warp takes a quarter of each job (copy runs, zero fill, V / offset staging) and arrives
// once on the stage's "full" barrier.  Two groups because a step's chain of barrier waits, copy issues and
// fences is latency-bound (~2000 clocks measured): two steps in flight double the rate.  Records arrive through
// a ring of SW_RING slots; the group working on step t requests record t + SW_LOOKAHEAD: having passed the
// "empty" wait of step t proves that the consumers, hence all producer warps, finished step t - 3, whose slot
// is the one overwritten.
template <class S, bool TENSOR>
__device__ __forceinline__ void sweep_producer(const sweep_args &a, const sweep_maps &maps, unsigned char *smem,
                                               uint32_t full0, uint32_t empty0, uint32_t rbar0, const unsigned char *recs,
                                               int nsteps, int ptid, double w0x3)
{
    constexpr int N = S::N, G = S::NGROUPS, GW = S::GW, GT = 32 * GW;   // GT threads per group
    constexpr int PPT = (S::NPT + GT - 1) / GT;   // tile points per thread (V and offsets)
    constexpr int HS = N / G;                     // a plane's store offsets are staged HS own steps after the plane itself
    constexpr int D = G == 1 ? 2 : 1;             // V and the offsets are fetched D own steps ahead (>= one full step period)
    const int group = ptid / GT, gtid = ptid % GT, lane = ptid & 31, pw = gtid >> 5;
    unsigned char *const ring = smem + (size_t)SW_STAGES * S::STAGE_BYTES;
    const uint32_t sbase = smem_u32(smem);
    auto request_rec = [&](int r) {   // one thread; preceded by a fence.proxy.async of that thread
        const uint32_t bar = rbar0 + 8u * (r % SW_RING);
        mbar_arrive_expect_tx(bar, S::REC_BYTES);
        bulk_g2s(smem_u32(ring) + (uint32_t)(r % SW_RING) * S::REC_BYTES, recs + (size_t)r * S::REC_BYTES, S::REC_BYTES, bar);
    };
    if (ptid == 0)
        for (int r = 0; r < SW_LOOKAHEAD && r < nsteps; ++r) request_rec(r);
    // this thread's jobs: copy run `myrun` (lanes 0..15 of each warp), a share of the zero fill, tile points gtid (+ 128)
    const int myrun = lane * GW + pw;
    // point p = (ty, tz): V at corner A row ty / 4, offsets at corner B row ty / 4 (4 tile rows per corner row)
    const uint32_t v_off0 = (uint32_t)(((gtid >> 6) * S::WZ) * SW_SLOT_BYTES + (gtid & 63) * 8);
    const uint32_t i_off0 = (uint32_t)(((gtid >> 6) * S::WZ + S::WZ - N) * SW_SLOT_BYTES + (gtid & 63) * 4);
    constexpr uint32_t NEXT_POINT = (GT / 64) * S::WZ * SW_SLOT_BYTES;   // point gtid + GT: GT / 64 corner rows further
    // stage = t mod SW_STAGES, record slot rs = t mod SW_RING and the barrier parities are re-derived from t where they are
    // needed instead of being carried: the producers run on 32 registers and a spilled V value would put the global-load
    // latency back on the per-step path (the first pass over the stages finds them free: parity 1)
    // V and the offsets of a plane are fetched one own step ahead of their use, and nothing touches the loaded value
    // until then, so that the global-load latency is not on the per-step path (adding 3 w_0 right after the load cost
    // ~1000 clocks per step: measured 0.136 -> 0.127 ms on config 2).  The store offsets of a plane's outputs are needed N steps later, when the x arm is
    // complete: this group staged that plane too (N is a multiple of the number of groups), so each thread simply
    // remembers its points' offsets for HS of its own steps and stages them with plane t.
    double vv[D][PPT];             // vv[0]: this own step's V, vv[D-1]: the value fetched last
    uint32_t hist[HS + D][PPT];    // offsets by age in own steps: hist[D-1] fetched last, hist[0] this step's, hist[HS] staged now
#pragma unroll
    for (int q = 0; q < PPT; ++q) {
#pragma unroll
        for (int d = 0; d < D; ++d) vv[d][q] = 0.0;
#pragma unroll
        for (int h = 0; h < HS + D; ++h) hist[h][q] = 0xffffffffu;
    }
    // shift the queues by one own step and fetch the V / offsets of the own step D - 1 ahead of the next one (record slot `slot`)
    auto advance_and_fetch = [&](int slot, bool have) {
#pragma unroll
        for (int q = 0; q < PPT; ++q) {
#pragma unroll
            for (int h = HS + D - 1; h > 0; --h) hist[h][q] = hist[h - 1][q];
#pragma unroll
            for (int d = 0; d + 1 < D; ++d) vv[d][q] = vv[d + 1][q];
            hist[0][q] = 0xffffffffu;
            vv[D - 1][q] = 0.0;
        }
        if (!have) return;
        const unsigned char *rp = ring + (size_t)slot * S::REC_BYTES;
        const uint32_t coff = *reinterpret_cast<const uint32_t *>(rp + SW_REC_HDR + 4);
#pragma unroll
        for (int q = 0; q < PPT; ++q) {
            const int p = gtid + GT * q;
            const int32_t ci = p < S::NPT ? *reinterpret_cast<const int32_t *>(rp + SW_REC_CIDX + p * 4) : -1;
            vv[D - 1][q] = ci >= 0 ? __ldg(a.vloc + ci) : -w0x3;   // consumed D own steps later, when 3 w_0 is added: no wait here
            hist[0][q] = ci >= 0 ? (uint32_t)ci * a.ncol + coff : 0xffffffffu;
        }
    };
    // prologue: the first D own steps' values (own step k of this group is step group + k * G)
#pragma unroll
    for (int d = 0; d < D; ++d) {
        const int tt = group + d * G;
        if (tt < nsteps) mbar_wait(rbar0 + 8u * (tt % SW_RING), (uint32_t)(tt / SW_RING) & 1u);
        advance_and_fetch(tt % SW_RING, tt < nsteps);
    }
    for (int t = group; t < nsteps; t += G) {
        const int stage = t % SW_STAGES, rs = t % SW_RING;
        const uint32_t eparity = ((uint32_t)(t / SW_STAGES) & 1u) ^ 1u;
        // everything the copies need is read from the record (present: fetch_v waited for it) BEFORE the wait for
        // the stage, so that the copies leave right after the consumers release it
        const unsigned char *rp = ring + (size_t)rs * S::REC_BYTES;
        const uint32_t sb = sbase + (uint32_t)stage * S::STAGE_BYTES;
        unsigned char *const sg = smem + (size_t)stage * S::STAGE_BYTES;
        const uint32_t bar = full0 + 8u * stage;
        const uint4 hdr = *reinterpret_cast<const uint4 *>(rp + SW_REC_HDR);   // {modes|flags, column offset, tx bytes 1-D, tx bytes 2-D}
        uint2 run = make_uint2(0u, 0u);
        if (lane < SW_MAXRUN / GW) run = *reinterpret_cast<const uint2 *>(rp + SW_REC_RUNS + myrun * 8);
        const uint32_t len = run.y >> 16, slot = run.y & 0xffffu;
        mbar_wait(empty0 + 8u * stage, eparity);
        const uint32_t nfill = (hdr.x >> HDR_NFILL_SHIFT) & 0xffu;
        if (nfill == HDR_NFILL_WHOLE) {
            // a piece's first planes: more slots to clear than the list holds -> the group clears the whole stage, and only
            // then (group barrier) may any of its warps issue the plane's copies
#pragma unroll 1
            for (uint32_t o = (uint32_t)gtid * 16u; o < (uint32_t)S::STAGE_BYTES; o += (uint32_t)GT * 16u)
                *reinterpret_cast<float4 *>(sg + o) = make_float4(0.f, 0.f, 0.f, 0.f);
            named_bar_sync(2 + group, GT);
        }
        fence_proxy_async();   // earlier generic accesses to this stage and to the record slot reused below (ordered before us by the barrier) before our async copies
        // ---- copy runs --------------------------------------------------------------------------------
        if (len) {
            if constexpr (!TENSOR) {
                bulk_g2s(sb + slot * SW_SLOT_BYTES, a.psi + (size_t)run.x * SW_C, len * SW_SLOT_BYTES, bar);
            } else {
                // largest box height (1, 2, 4, 8, 16 or 24) not above len; a second, overlapping box covers the rest
                const int lg = len >= 24 ? 5 : 31 - __clz((int)len);
                const uint32_t p = len >= 24 ? 24u : 1u << lg;
                tensor_g2s(sb + slot * SW_SLOT_BYTES, &maps.box[lg], (int)hdr.y, (int)run.x, bar);
                if (p < len)
                    tensor_g2s(sb + (slot + len - p) * SW_SLOT_BYTES, &maps.box[lg], (int)hdr.y, (int)(run.x + len - p), bar);
            }
        }
        if (gtid == 0 && t + SW_LOOKAHEAD < nsteps) request_rec(t + SW_LOOKAHEAD);
        // ---- zero fill: the record lists the slots of the [WY][WZ] grid that must be cleared (lattice point outside the
        //      mesh and the buffer does not already hold zeros there): a warp takes 16 list entries, a quarter-warp 4 of
        //      them (one 8-byte load), each slot cleared with 8 conflict-free 16-byte stores.  No search, no dependent
        //      branches: walking a bitmap cost 800..3500 clocks per step, every word a dependent load behind the consumers' traffic.
        {
            constexpr int EPQ = SW_MAXFILL / GW / 4;   // list entries per quarter-warp: 4 (one 8-byte load) or 2 (one 4-byte load)
            const uint32_t e0 = (uint32_t)(pw * (SW_MAXFILL / GW) + EPQ * (lane >> 3));
            if (e0 < nfill && nfill != HDR_NFILL_WHOLE) {
                uint32_t ent[2];
                if constexpr (EPQ == 4) {
                    const uint2 four = *reinterpret_cast<const uint2 *>(rp + SW_REC_FLIST + 2 * e0);
                    ent[0] = four.x, ent[1] = four.y;
                } else {
                    ent[0] = *reinterpret_cast<const uint32_t *>(rp + SW_REC_FLIST + 2 * e0), ent[1] = 0;
                }
                unsigned char *const dst = sg + (lane & 7) * 16;
#pragma unroll
                for (int i = 0; i < EPQ; ++i)
                    if (e0 + i < nfill)
                        *reinterpret_cast<float4 *>(dst + (size_t)((ent[i >> 1] >> (16 * (i & 1))) & 0xffffu) * SW_SLOT_BYTES) = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
        // ---- V of the tile's own points (output planes only) and the store offsets of plane t - N ------------
#pragma unroll
        for (int q = 0; q < PPT; ++q) {
            if (gtid + GT * q < S::NPT) {
                if (hdr.x & HDR_OUTPUT_PLANE)   // 3 w_0 + V: the whole diagonal coefficient
                    *reinterpret_cast<double *>(sg + v_off0 + q * NEXT_POINT) = vv[0][q] + w0x3;
                *reinterpret_cast<uint32_t *>(sg + i_off0 + q * NEXT_POINT) = hist[HS + D - 1][q];
            }
        }
        if (gtid == 0) *reinterpret_cast<uint2 *>(sg + S::HDR_OFF) = make_uint2(hdr.x, hdr.y);
        __syncwarp();
        // one arrival per warp; the group's first thread also announces the bytes of all the group's copies (the
        // count may run negative until then: the phase cannot complete before this arrival)
        if (lane == 0) {
            if (pw == 0)
                mbar_arrive_expect_tx(bar, TENSOR ? hdr.w : hdr.z);
            else
                mbar_arrive(bar);
        }
        {   // the queues move on by one own step; fetch for the own step D ahead (its record was requested SW_LOOKAHEAD steps before it)
            const int tn = t + D * G;
            if (tn < nsteps) mbar_wait(rbar0 + 8u * (tn % SW_RING), (uint32_t)(tn / SW_RING) & 1u);
            advance_and_fetch(tn % SW_RING, tn < nsteps);
        }
    }
}

// ---- consumer warps: the arithmetic ----------------------------------------------------------------
// tensor memory, one patch row: [ring slot t mod N][4 doubles]; loaded whole (N x 8 words), stored one slot at a time
template <int N>
__device__ __forceinline__ void tm_ld_row(uint32_t taddr, uint32_t (&r)[N * 8])
{
    static_assert(N == 4 || N == 6, "tensor-memory row shapes");
    uint32_t(&lo)[32] = reinterpret_cast<uint32_t(&)[32]>(r[0]);
    tm_ld32(taddr, lo);
    if constexpr (N == 6) {
        uint32_t(&hi)[16] = reinterpret_cast<uint32_t(&)[16]>(r[32]);
        tm_ld16(taddr + 32, hi);
    }
}
template <int N>
__device__ __forceinline__ void tm_wait_row(uint32_t (&r)[N * 8])
{
    uint32_t(&lo)[32] = reinterpret_cast<uint32_t(&)[32]>(r[0]);
    if constexpr (N == 6) {
        uint32_t(&hi)[16] = reinterpret_cast<uint32_t(&)[16]>(r[32]);
        tm_wait_ld16(hi);
    }
    tm_wait_ld32(lo);
}

template <class S, bool HALF>
__device__ __forceinline__ void sweep_consumer(const sweep_args &a, const rs_weights &w, const unsigned char *smem,
                                               uint32_t full0, uint32_t empty0, uint32_t tmem_base, int nsteps, int tid,
                                               long long *step_clock)
{
    constexpr int N = S::N, PY = S::PY, PZ = SW_PZ, WZ = S::WZ;
    const int lane = tid & 31, warp = tid >> 5;
    const int c = tid & 15, patch = tid >> 4, py = patch >> 2, pz = patch & 3;
    const int ty0 = PY * py;   // first tile row of the patch
    // this thread's TMEM lane (its warp's quarter) and the column range of its warp:
    // [patch row j][ring slot t mod N][i]: centre values of the last N planes (doubles)
    const uint32_t t_in = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(warp >> 2) * (PY * S::ROW_WORDS);

    const uint32_t b0 = (uint32_t)(((N + ty0) * WZ + PZ * pz) * SW_SLOT_BYTES + c * 8);   // patch row 0, window slot 0
    // V (corner A) and store offsets (corner B): 4 tile rows per corner row, PY divides 4
    const uint32_t vrow = (uint32_t)(((ty0 >> 2) * WZ) * SW_SLOT_BYTES + ((ty0 & 3) * SW_TZ + PZ * pz) * 8);
    const uint32_t irow = (uint32_t)(((ty0 >> 2) * WZ + WZ - N) * SW_SLOT_BYTES + ((ty0 & 3) * SW_TZ + PZ * pz) * 4);

    double acc[N][PY][PZ];   // pending outputs: acc[t mod N] belongs to plane t
#pragma unroll
    for (int k = 0; k < N; ++k)
#pragma unroll
        for (int j = 0; j < PY; ++j)
#pragma unroll
            for (int i = 0; i < PZ; ++i) acc[k][j][i] = 0.0;
    int stage = 0;
    uint32_t parity = 0;
    double *const hp = a.hpsi + c;

    for (int t0 = 0; t0 < nsteps; t0 += N) {
#pragma unroll
        for (int PH = 0; PH < N; ++PH) {
            const int t = t0 + PH;
            if (t >= nsteps) break;
            tm_wait_st();
            mbar_wait(full0 + 8u * stage, parity);
            const unsigned char *sp = smem + (size_t)stage * S::STAGE_BYTES;
            const uint2 hdr = *reinterpret_cast<const uint2 *>(sp + S::HDR_OFF);   // {modes | flags, column offset}
            const int mode = (int)((hdr.x >> (2 * warp)) & 3u);
            const double *pb = reinterpret_cast<const double *>(sp + b0);

            // store offsets of the outputs this step completes (plane t - N), staged by the producer; -1: none
            uint32_t io[PY * PZ];
#pragma unroll
            for (int j = 0; j < PY; ++j) {
                const uint4 q = *reinterpret_cast<const uint4 *>(sp + irow + j * 64);
                io[4 * j] = q.x, io[4 * j + 1] = q.y, io[4 * j + 2] = q.z, io[4 * j + 3] = q.w;
            }
            if constexpr (HALF) {   // 8-column block: the upper lanes hold the zero-filled columns and own no output
                if (c >= SW_C / 2) {
#pragma unroll
                    for (int q = 0; q < PY * PZ; ++q) io[q] = 0xffffffffu;
                }
            }

            if (mode == MODE_FULL) {
                double ctr[PY][PZ];
#pragma unroll
                for (int j = 0; j < PY; ++j) {
                    uint32_t pw[N * 8];   // centre values of planes t-1 .. t-N of this patch row
                    tm_ld_row<N>(t_in + j * S::ROW_WORDS, pw);
                    double v[PZ + 2 * N];
#pragma unroll
                    for (int tt = 0; tt < PZ + 2 * N; ++tt)
                        v[tt] = pb[(j * WZ + tt) * SW_C];
                    const double2 va = *reinterpret_cast<const double2 *>(sp + vrow + j * 128);
                    const double2 vb = *reinterpret_cast<const double2 *>(sp + vrow + j * 128 + 16);
                    const double vv[4] = {va.x, va.y, vb.x, vb.y};
                    double s[PZ];
#pragma unroll
                    for (int i = 0; i < PZ; ++i) {
                        const double ce = v[N + i];
                        ctr[j][i] = ce;
#pragma unroll
                        for (int k = 1; k < N; ++k) acc[(PH + N - k) % N][j][i] = fma(w.w[k], ce, acc[(PH + N - k) % N][j][i]);
                        const double out = fma(w.w[N], ce, acc[PH][j][i]);
                        store_if_valid(hp, io[4 * j + i], out);
                        s[i] = vv[i] * ce;   // vv = 3 w_0 + V, formed by the producer
#pragma unroll
                        for (int k = 1; k <= N; ++k) {
                            s[i] = fma(w.w[k], v[N + i + k], s[i]);
                            s[i] = fma(w.w[k], v[N + i - k], s[i]);
                        }
                    }
                    // backward half of the x arm from tensor memory, then park this row's centre values
                    tm_wait_row<N>(pw);
#pragma unroll
                    for (int i = 0; i < PZ; ++i) {
#pragma unroll
                        for (int k = 1; k <= N; ++k) {
                            const int sl = (PH + N - k) % N;
                            s[i] = fma(w.w[k], words2double(pw[sl * 8 + 2 * i], pw[sl * 8 + 2 * i + 1]), s[i]);
                        }
                        acc[PH][j][i] = s[i];
                    }
                    uint32_t cw[8];
#pragma unroll
                    for (int i = 0; i < PZ; ++i) {
                        cw[2 * i] = (uint32_t)__double2loint(ctr[j][i]);
                        cw[2 * i + 1] = (uint32_t)__double2hiint(ctr[j][i]);
                    }
                    tm_st8(t_in + j * S::ROW_WORDS + PH * 8, cw);
                }
                // y arms: rows ty0-N .. ty0+PY-1+N of the patch's 4 z columns
#pragma unroll
                for (int i = 0; i < PZ; ++i) {
                    double u[PY + 2 * N];
#pragma unroll
                    for (int tt = 0; tt < PY + 2 * N; ++tt)
                        u[tt] = (tt >= N && tt < N + PY) ? ctr[tt - N][i] : pb[((tt - N) * WZ + N + i) * SW_C];
#pragma unroll
                    for (int j = 0; j < PY; ++j)
#pragma unroll
                        for (int k = 1; k <= N; ++k) {
                            acc[PH][j][i] = fma(w.w[k], u[N + j + k], acc[PH][j][i]);
                            acc[PH][j][i] = fma(w.w[k], u[N + j - k], acc[PH][j][i]);
                        }
                }
            } else if (mode == MODE_CENTRE) {
                // centre-only plane (warm-up / tail of a work item): it feeds the x arms of its neighbours
#pragma unroll
                for (int j = 0; j < PY; ++j) {
                    uint32_t cw[8];
#pragma unroll
                    for (int i = 0; i < PZ; ++i) {
                        const double ce = pb[(j * WZ + N + i) * SW_C];
#pragma unroll
                        for (int k = 1; k < N; ++k) acc[(PH + N - k) % N][j][i] = fma(w.w[k], ce, acc[(PH + N - k) % N][j][i]);
                        const double out = fma(w.w[N], ce, acc[PH][j][i]);
                        store_if_valid(hp, io[4 * j + i], out);
                        acc[PH][j][i] = 0.0;
                        cw[2 * i] = (uint32_t)__double2loint(ce);
                        cw[2 * i + 1] = (uint32_t)__double2hiint(ce);
                    }
                    tm_st8(t_in + j * S::ROW_WORDS + PH * 8, cw);
                }
            } else {
                // no mesh point of this warp's region in plane t: all centre values are zero
                uint32_t cw[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) cw[q] = 0u;
#pragma unroll
                for (int j = 0; j < PY; ++j) {
#pragma unroll
                    for (int i = 0; i < PZ; ++i) {
                        store_if_valid(hp, io[4 * j + i], acc[PH][j][i]);
                        acc[PH][j][i] = 0.0;
                    }
                    tm_st8(t_in + j * S::ROW_WORDS + PH * 8, cw);
                }
            }
            // this warp has read everything it needs from the stage
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8u * stage);
            if (tid == 0 && step_clock) step_clock[t] = clock64();
            if (++stage == SW_STAGES) {
                stage = 0;
                parity ^= 1u;
            }
        }
    }
    tm_wait_st();
}

template <int REGS>
__device__ __forceinline__ void setmaxnreg_inc()
{
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(REGS));
}
template <int REGS>
__device__ __forceinline__ void setmaxnreg_dec()
{
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(REGS));
}

template <class S, bool TENSOR, bool HALF = false>
__global__ void __launch_bounds__(S::THREADS, 1)
sweep_kernel(const __grid_constant__ sweep_args a, const __grid_constant__ rs_weights w, const __grid_constant__ sweep_maps maps)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint64_t full_bar[SW_STAGES];
    __shared__ uint64_t empty_bar[SW_STAGES];
    __shared__ uint64_t rec_bar[SW_RING];
    __shared__ uint32_t tmem_base_s;

    // consumer warps take the low warp ids, producer warps the high ones (the other way round measured the same)
    const int tid = threadIdx.x, warp = tid >> 5;
    const int ctid = tid < S::CONSUMERS ? tid : -1;
    const int ptid = tid - S::CONSUMERS;
    const int2 item = a.items[blockIdx.x];
    const int nsteps = item.y;
    const long long clock0 = clock64();

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < SW_STAGES; ++s) {
            mbar_init(smem_u32(&full_bar[s]), S::GW);   // the warps of the producer group that stages the step
            mbar_init(smem_u32(&empty_bar[s]), S::NCW);
        }
#pragma unroll
        for (int s = 0; s < SW_RING; ++s) mbar_init(smem_u32(&rec_bar[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 0) {   // first consumer warp
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&tmem_base_s)),
                     "n"(SW_TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");

    // register re-split: THREADS x LAUNCH_REGS at launch -> PRODUCERS x PROD_REGS + CONSUMERS x CONS_REGS; the pool that
    // setmaxnreg.inc draws from holds only what setmaxnreg.dec released, so the increase must not exceed the release
    static_assert(S::CONSUMERS * (S::CONS_REGS - S::LAUNCH_REGS) <= S::PRODUCERS * (S::LAUNCH_REGS - S::PROD_REGS), "register pool");
    if (ctid < 0) {
        setmaxnreg_dec<S::PROD_REGS>();
        sweep_producer<S, TENSOR>(a, maps, smem, smem_u32(&full_bar[0]), smem_u32(&empty_bar[0]), smem_u32(&rec_bar[0]),
                                  a.recs + (size_t)item.x * S::REC_BYTES, nsteps, ptid, 3.0 * w.w[0]);
    } else {
        setmaxnreg_inc<S::CONS_REGS>();
        sweep_consumer<S, HALF>(a, w, smem, smem_u32(&full_bar[0]), smem_u32(&empty_bar[0]), tmem_base_s, nsteps, ctid,
                          a.step_clock ? a.step_clock + item.x : nullptr);
        named_bar_sync(1, S::CONSUMERS);
        if (ctid == 0 && a.cycles) a.cycles[blockIdx.x] = clock64() - clock0;
        if (ctid < 32)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base_s), "n"(SW_TMEM_COLS) : "memory");
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host: work pieces, their assignment to CTAs, and the per-step records
// ---------------------------------------------------------------------------------------------
namespace {
enum { VARIANT_N4 = 0, VARIANT_N6 = 1, VARIANT_NONE = -1 };
// Block widths (real columns): multiples of 16 are processed 16 columns at a time; 8 columns run as HALF a slice -- the
// tensor-map boxes are 16 columns wide whatever the block's width, the copy unit zero-fills the 8 columns that lie
// outside the row, and the consumer lanes of those columns compute on zeros and store nothing.
constexpr int SW_HALF = SW_C / 2;
bool sweep_width_ok(int ncol) { return ncol == SW_HALF || (ncol >= SW_C && ncol % SW_C == 0); }
int sweep_nchunks(int ncol) { return ncol < SW_C ? 1 : ncol / SW_C; }
int sweep_variant(int n) { return n == 4 ? VARIANT_N4 : n == 6 ? VARIANT_N6 : VARIANT_NONE; }
shape_rt variant_shape(int variant) { return variant == VARIANT_N6 ? shape_of<shape_n6>() : shape_of<shape_n4>(); }
}  // namespace

namespace {

// modelled cost of a step, in units of a step whose 8 warps are all in full mode.  Least-squares fit of the per-CTA
// clock counts of the kernel itself (rs_sweep_stats; config 2, B = 16 on B200, rms error 3 %):
//   clocks = 1976 steps + 124 full warp-steps + 2484 pieces   (a full step: 1976 + 8 x 124 = 2968 clocks)
// i.e. two thirds of a step's time does not depend on how many warps compute: it is the latency of the
// release -> stage -> copy -> consume chain through the 3 stage buffers.
constexpr double COST_STEP_FIXED = 0.666, COST_FULL_WARP = 0.042, COST_CENTRE_WARP = 0.006, COST_PIECE = 0.84;
constexpr double COST_EMPTY_STEP = COST_STEP_FIXED;

struct tile_geometry {
    const rs_mesh *m;
    shape_rt sh;
    int nx, ny, nz, nty, ntz;
    int32_t point(int x, int y, int z) const
    {
        if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) return -1;
        return m->dense2point[rs_dense_index(m, x, y, z)];
    }
    // 2 bits per warp for plane x of tile (iy, iz): which warps' PY x 8 regions hold a mesh point
    // (a warp = two patches next to each other in z: patch rows PY * (w / 2) .., z columns 8 * (w % 2) ..)
    uint32_t warp_modes(int iy, int iz, int x, int mode) const
    {
        uint32_t hdr = 0;
        for (int wq = 0; wq < sh.NCW; ++wq) {
            bool any = false;
            for (int y = sh.PY * (wq >> 1); y < sh.PY * (wq >> 1) + sh.PY && !any; ++y)
                for (int z = 8 * (wq & 1); z < 8 * (wq & 1) + 8 && !any; ++z) any = point(x, iy * sh.TY + y, iz * SW_TZ + z) >= 0;
            if (any) hdr |= (uint32_t)mode << (2 * wq);
        }
        return hdr;
    }
};

double step_cost(uint32_t modes, int ncw)
{
    double c = COST_STEP_FIXED;
    for (int q = 0; q < ncw; ++q) {
        const uint32_t md = (modes >> (2 * q)) & 3u;
        c += (md == MODE_FULL ? COST_FULL_WARP : md == MODE_CENTRE ? COST_CENTRE_WARP : 0.0) * 8.0 / ncw;
    }
    return c;
}

}  // namespace

bool rs_sweep_build_host(const rs_mesh *m, int n, int ncol, int max_planes, int nctas, rs_sweep_host &out,
                         const rs_sweep_costs *measured, const std::vector<std::vector<rs_sweep_piece>> *given_pieces)
{
    const int variant = sweep_variant(n);
    if (variant == VARIANT_NONE || !sweep_width_ok(ncol) || nctas < 1) return false;
    const shape_rt sh = variant_shape(variant);
    const int N = sh.N, TY = sh.TY, TZ = SW_TZ, WY = sh.WY, WZ = sh.WZ;
    tile_geometry g{m, sh, m->dims[0], m->dims[1], m->dims[2], (m->dims[1] + TY - 1) / TY, (m->dims[2] + TZ - 1) / TZ};
    const int nx = g.nx, nchunks = sweep_nchunks(ncol);
    out = rs_sweep_host();
    out.rec_bytes = sh.rec_bytes;

    // ---- cost of every (tile, plane) as a full step; 0 where the tile has no mesh point in the plane ----
    std::vector<double> fcost((size_t)g.nty * g.ntz * nx, 0.0), ccost((size_t)g.nty * g.ntz * nx, 0.0);
    for (int iy = 0; iy < g.nty; ++iy)
        for (int iz = 0; iz < g.ntz; ++iz)
            for (int x = 0; x < nx; ++x) {
                const uint32_t mf = g.warp_modes(iy, iz, x, MODE_FULL);
                if (mf) {
                    fcost[((size_t)iy * g.ntz + iz) * nx + x] = step_cost(mf, sh.NCW);
                    ccost[((size_t)iy * g.ntz + iz) * nx + x] = step_cost(g.warp_modes(iy, iz, x, MODE_CENTRE), sh.NCW);
                }
            }
    // measured step costs (rs_hamiltonian_autotune), relative to the mean output step, replace the model where present
    double cost_piece = COST_PIECE, cost_empty = COST_EMPTY_STEP;
    if (measured && measured->unit > 0.0 && measured->full.size() == fcost.size()) {
        double ratio_sum = 0.0;   // measured / model over the measured cells: scales the model for the others
        int64_t ratio_n = 0;
        for (size_t q = 0; q < fcost.size(); ++q)
            if (fcost[q] > 0.0 && measured->full[q] > 0.f) ratio_sum += measured->full[q] / measured->unit / fcost[q], ++ratio_n;
        const double scale = ratio_n ? ratio_sum / ratio_n : 1.0;
        for (size_t q = 0; q < fcost.size(); ++q)
            if (fcost[q] > 0.0) fcost[q] = measured->full[q] > 0.f ? measured->full[q] / measured->unit : fcost[q] * scale;
        cost_empty = measured->halo / measured->unit;
        for (double &c : ccost)
            if (c > 0.0) c = cost_empty;
        cost_piece = 0.0;   // a piece's start-up is part of its measured steps
    }
    auto halo_cost = [&](int iy, int iz, int xa, int xb) {   // the 2 N centre-only steps around [xa, xb) + the piece's own overhead
        double c = cost_piece;
        const double *cc = &ccost[((size_t)iy * g.ntz + iz) * nx];
        for (int k = 1; k <= N; ++k) {
            c += (xa - k >= 0 && cc[xa - k] > 0.0) ? cc[xa - k] : cost_empty;
            c += (xb + k - 1 < nx && cc[xb + k - 1] > 0.0) ? cc[xb + k - 1] : cost_empty;
        }
        return c;
    };
    auto range_cost = [&](int iy, int iz, int xa, int xb) {
        double c = 0.0;
        const double *fc = &fcost[((size_t)iy * g.ntz + iz) * nx];
        for (int x = xa; x < xb; ++x) c += fc[x] > 0.0 ? fc[x] : cost_empty;
        return c;
    };

    // ---- work items in execution order: slab by slab, column slice by column slice, tile by tile -------
    std::vector<rs_sweep_piece> items;
    double total = 0.0;
    for (int xs = 0; xs < nx; xs += max_planes) {
        const int xe = std::min(nx, xs + max_planes);
        for (int ch = 0; ch < nchunks; ++ch)
            for (int iy = 0; iy < g.nty; ++iy)
                for (int iz = 0; iz < g.ntz; ++iz) {
                    const double *fc = &fcost[((size_t)iy * g.ntz + iz) * nx];
                    int xa = -1, xb = -1;
                    for (int x = xs; x < xe; ++x)
                        if (fc[x] > 0.0) {
                            if (xa < 0) xa = x;
                            xb = x + 1;
                        }
                    if (xa < 0) continue;
                    items.push_back({iy, iz, xa, xb, ch});
                    total += range_cost(iy, iz, xa, xb) + halo_cost(iy, iz, xa, xb);
                }
    }
    // ---- deal them out: always to the least-loaded CTA; an item that would overshoot the common finish
    //      line is split in x, the rest goes back to the head of the queue ---------------------------------
    std::vector<double> load;
    auto deal = [&](double finish, std::vector<std::vector<rs_sweep_piece>> &pieces) -> double {
        pieces.assign(nctas, {});
        load.assign(nctas, 0.0);
        std::vector<char> closed(nctas, 0);   // CTAs that cannot take another piece without overshooting
        const int MIN_SPLIT = m->opt.min_split < 1 ? 1 : m->opt.min_split;   // output planes: below this the 2 N halo steps dominate
        auto least_loaded = [&](bool open_only) {
            int best = -1;
            for (int c = 0; c < nctas; ++c)
                if ((!open_only || !closed[c]) && (best < 0 || load[c] < load[best])) best = c;
            return best;
        };
        for (size_t q = 0; q < items.size(); ++q) {
            rs_sweep_piece it = items[q];
            for (;;) {
                int cta = least_loaded(true);
                const double whole = range_cost(it.iy, it.iz, it.xa, it.xb) + halo_cost(it.iy, it.iz, it.xa, it.xb);
                if (cta < 0) {   // every CTA is at the finish line: the least loaded takes the overshoot
                    cta = least_loaded(false);
                    pieces[cta].push_back(it);
                    load[cta] += whole;
                    break;
                }
                if (load[cta] + whole <= finish) {
                    pieces[cta].push_back(it);
                    load[cta] += whole;
                    break;
                }
                // largest prefix [xa, xsplit) that still fits, leaving at least MIN_SPLIT planes on either side
                int xsplit = it.xa;
                double c = halo_cost(it.iy, it.iz, it.xa, it.xb);
                const double *fc = &fcost[((size_t)it.iy * g.ntz + it.iz) * nx];
                while (xsplit < it.xb - MIN_SPLIT) {
                    const double cx = fc[xsplit] > 0.0 ? fc[xsplit] : cost_empty;
                    if (load[cta] + c + cx > finish) break;
                    c += cx;
                    ++xsplit;
                }
                if (xsplit - it.xa < MIN_SPLIT) {
                    closed[cta] = 1;
                    continue;
                }
                rs_sweep_piece head = it;
                head.xb = xsplit;
                pieces[cta].push_back(head);
                load[cta] += range_cost(head.iy, head.iz, head.xa, head.xb) + halo_cost(head.iy, head.iz, head.xa, head.xb);
                it.xa = xsplit;
            }
        }
        return *std::max_element(load.begin(), load.end());
    };
    // the lowest common finish line that the dealing meets without overshoot (bisection)
    double lo = total / nctas, hi = lo * 1.05 + 2.0;
    std::vector<std::vector<rs_sweep_piece>> trial;
    while (deal(hi, trial) > hi) hi = hi * 1.25 + 2.0;
    for (int it = 0; it < 14; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (deal(mid, trial) <= mid)
            hi = mid;
        else
            lo = mid;
    }
    deal(hi, out.pieces);
    if (given_pieces && (int)given_pieces->size() == nctas) {   // a refined dealing (rs_hamiltonian_autotune) replaces the dealt one
        out.pieces = *given_pieces;
        for (int c = 0; c < nctas; ++c) {
            load[c] = 0.0;
            for (const rs_sweep_piece &pc : out.pieces[c]) load[c] += range_cost(pc.iy, pc.iz, pc.xa, pc.xb) + halo_cost(pc.iy, pc.iz, pc.xa, pc.xb);
        }
    }
    out.load = load;
    for (double l : load) {
        out.cost_max = std::max(out.cost_max, l);
        out.cost_mean += l / nctas;
    }

    // ---- records: one per (CTA, step) ----------------------------------------------------------------
    enum { UNKNOWN = 0, ZERO = 1, DATA = 2 };
    std::vector<uint8_t> state((size_t)SW_STAGES * WY * WZ);
    out.items.resize(nctas);
    for (int cta = 0; cta < nctas; ++cta) {
        std::fill(state.begin(), state.end(), (uint8_t)UNKNOWN);   // shared memory of a starting CTA is arbitrary
        const int64_t first = out.nrec;
        int step = 0;                                               // stage of a step = step mod SW_STAGES, as in the kernel
        for (const rs_sweep_piece &pc : out.pieces[cta]) {
            const int y0 = pc.iy * TY, z0 = pc.iz * TZ;
            const int nsteps = (pc.xb - pc.xa) + 2 * N;
            for (int s = 0; s < nsteps; ++s, ++step) {
                const int p = pc.xa - N + s;
                const bool full = s >= N && s < nsteps - N;
                out.recs.resize((size_t)(out.nrec + 1) * sh.rec_bytes, 0);
                unsigned char *rec = out.recs.data() + (size_t)out.nrec * sh.rec_bytes;
                uint2 *runs = reinterpret_cast<uint2 *>(rec + SW_REC_RUNS);
                uint32_t *fill = reinterpret_cast<uint32_t *>(rec + SW_REC_FILL);
                uint32_t *hdrp = reinterpret_cast<uint32_t *>(rec + SW_REC_HDR);
                int32_t *cidx = reinterpret_cast<int32_t *>(rec + SW_REC_CIDX);
                uint8_t *st = &state[(size_t)(step % SW_STAGES) * WY * WZ];
                // copy runs, and zero-fill bits for the slots this plane reads that are outside the mesh and
                // do not already hold zeros from an earlier plane staged in the same buffer
                int nrun = 0;
                uint32_t tx1 = 0, tx2 = 0;
                uint32_t datamask[20] = {};   // slots that receive data from this plane's copy runs
                for (int r = full ? 0 : N; r < (full ? WY : N + TY); ++r) {
                    const bool halo_row = r < N || r >= N + TY;
                    const int zlo = (halo_row || !full) ? N : 0, zhi = (halo_row || !full) ? N + TZ : WZ;
                    int run_start = -1;
                    for (int zp = zlo; zp <= zhi; ++zp) {
                        const int32_t idx = zp < zhi ? g.point(p, y0 - N + r, z0 - N + zp) : -1;
                        if (idx >= 0) {
                            if (run_start < 0) run_start = zp;
                            st[r * WZ + zp] = DATA;
                            datamask[(r * WZ + zp) >> 5] |= 1u << ((r * WZ + zp) & 31);
                        } else {
                            if (run_start >= 0) {
                                if (nrun >= SW_MAXRUN) return false;
                                const int32_t firstp = g.point(p, y0 - N + r, z0 - N + run_start);
                                const uint32_t len = (uint32_t)(zp - run_start);
                                runs[nrun++] = make_uint2((uint32_t)firstp, (uint32_t)(r * WZ + run_start) | (len << 16));
                                uint32_t box = 24;
                                if (len < 24)
                                    for (box = 1; box * 2 <= len; box *= 2) {}
                                tx1 += len * SW_SLOT_BYTES;
                                tx2 += (box < len ? 2 * box : box) * SW_SLOT_BYTES;
                                run_start = -1;
                            }
                            if (zp < zhi && st[r * WZ + zp] != ZERO) {
                                fill[(r * WZ + zp) >> 5] |= 1u << ((r * WZ + zp) & 31);
                                st[r * WZ + zp] = ZERO;
                            }
                        }
                    }
                }
                // the clear list: the set bits of the bitmap in ascending order; if there are more than the list holds, the
                // kernel clears the WHOLE stage before the copies: then the bitmap names every slot without data
                uint32_t nfill = 0;
                uint16_t *flist = reinterpret_cast<uint16_t *>(rec + SW_REC_FLIST);
                for (int sl = 0; sl < WY * WZ; ++sl) nfill += (fill[sl >> 5] >> (sl & 31)) & 1u;
                if (nfill > (uint32_t)SW_MAXFILL) {
                    for (int sl = 0; sl < WY * WZ; ++sl) {
                        if (st[sl] == DATA && /* staged by THIS plane */ ((datamask[sl >> 5] >> (sl & 31)) & 1u)) continue;
                        fill[sl >> 5] |= 1u << (sl & 31);
                        st[sl] = ZERO;
                    }
                    nfill = HDR_NFILL_WHOLE;
                } else {
                    uint32_t q = 0;
                    for (int sl = 0; sl < WY * WZ; ++sl)
                        if ((fill[sl >> 5] >> (sl & 31)) & 1u) flist[q++] = (uint16_t)sl;
                }
                hdrp[0] = g.warp_modes(pc.iy, pc.iz, p, full ? MODE_FULL : MODE_CENTRE) | (full ? HDR_OUTPUT_PLANE : 0u) |
                          (nfill << HDR_NFILL_SHIFT);
                hdrp[1] = (uint32_t)(pc.chunk * SW_C);
                hdrp[2] = tx1;
                hdrp[3] = tx2;
                out.rec_cell.push_back(full && p >= 0 && p < nx ? (int32_t)(((size_t)pc.iy * g.ntz + pc.iz) * nx + p) : -1);
                for (int y = 0; y < TY; ++y)
                    for (int z = 0; z < TZ; ++z) cidx[y * TZ + z] = full ? g.point(p, y0 + y, z0 + z) : -1;
                ++out.nrec;
            }
        }
        out.items[cta] = make_int2((int)first, step);
    }
    return true;
}

bool rs_sweep_supported(const rs_mesh *m, int n, int ncol)
{
    return m->ordering == RS_ORDER_LEX && !m->periodic && sweep_variant(n) != VARIANT_NONE && sweep_width_ok(ncol) &&
           (uint64_t)(m->np + 1) * (uint64_t)ncol < 0xffffffffull;   // store offsets are 32-bit element offsets
}

static int sweep_nctas(const rs_mesh *m) { return m->opt.ctas > 0 ? m->opt.ctas : (m->sm_count > 0 ? m->sm_count : 148); }
static int clamp_planes(int v) { return v < 4 ? 4 : v; }

template <class S>
static cudaError_t set_smem()
{
    cudaError_t e = cudaFuncSetAttribute(sweep_kernel<S, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sweep_kernel<S, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(sweep_kernel<S, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::SMEM);
}

template <class S>
static void launch_shape(bool tensor, unsigned grid, cudaStream_t st, const sweep_args &a, const rs_weights &w, const sweep_maps &maps)
{
    if (a.ncol == (uint32_t)SW_HALF)
        sweep_kernel<S, true, true><<<grid, S::THREADS, S::SMEM, st>>>(a, w, maps);
    else if (tensor)
        sweep_kernel<S, true><<<grid, S::THREADS, S::SMEM, st>>>(a, w, maps);
    else
        sweep_kernel<S, false><<<grid, S::THREADS, S::SMEM, st>>>(a, w, maps);
}

static rs_status get_tables(rs_mesh *m, int n, int ncol, const rs_sweep_tables **out)
{
    const auto key = std::make_pair(n * 16 + sweep_variant(n), ncol);
    auto f = m->sweep.find(key);
    if (f == m->sweep.end()) {
        rs_sweep_host h;
        rs_sweep_tables tb;
        const auto mc = m->sweep_costs.find(key);
        const bool tuned = mc != m->sweep_costs.end();
        const auto gp = m->sweep_pieces.find(key);
        tb.ok = rs_sweep_build_host(m, n, ncol, clamp_planes(tuned ? m->opt.planes_tuned : m->opt.planes), sweep_nctas(m), h, tuned ? &mc->second : nullptr,
                                    gp != m->sweep_pieces.end() ? &gp->second : nullptr);
        if (tb.ok) {
            tb.nitems = (int64_t)h.items.size();
            tb.nrec = h.nrec;
            auto up = [&](void **d, const void *src, size_t bytes) -> cudaError_t {
                cudaError_t e = cudaMalloc(d, bytes ? bytes : 16);
                if (e != cudaSuccess || bytes == 0) return e;
                tb.bytes += (int64_t)bytes;
                return cudaMemcpy(*d, src, bytes, cudaMemcpyHostToDevice);
            };
            RS_CUDA_TRY(up((void **)&tb.d_items, h.items.data(), h.items.size() * sizeof(int2)));
            RS_CUDA_TRY(up((void **)&tb.d_recs, h.recs.data(), h.recs.size()));
            RS_CUDA_TRY(cudaMalloc((void **)&tb.d_step_clock, (size_t)(h.nrec + 1) * sizeof(long long)));
            tb.host_items = h.items;
            tb.pieces = h.pieces;
            tb.rec_cell = h.rec_cell;
            RS_CUDA_TRY(cudaMalloc((void **)&tb.d_cycles, (h.items.size() + 2048) * sizeof(long long)));
            RS_CUDA_TRY(cudaMemset(tb.d_cycles, 0, (h.items.size() + 2048) * sizeof(long long)));
            tb.variant = sweep_variant(n);
            for (size_t c = 0; c < h.items.size(); ++c) {
                int64_t nfull = 0;
                for (int t = 0; t < h.items[c].y; ++t) {
                    const uint32_t hd = *reinterpret_cast<const uint32_t *>(h.recs.data() + (size_t)(h.items[c].x + t) * h.rec_bytes + SW_REC_HDR);
                    for (int wq = 0; wq < 8; ++wq) nfull += ((hd >> (2 * wq)) & 3u) == MODE_FULL;
                }
                tb.host_stats.insert(tb.host_stats.end(), {(int64_t)h.items[c].y, (int64_t)h.pieces[c].size(), (int64_t)(h.load[c] * 1000), nfull});
            }
            RS_CUDA_TRY(set_smem<shape_n4>());
            RS_CUDA_TRY(set_smem<shape_n6>());
        }
        f = m->sweep.emplace(key, tb).first;
    }
    *out = &f->second;
    return RS_OK;
}

// psi viewed as a [np + 1][ncol] fp64 tensor; one map per box height (1, 2, 4, 8, 16, 24 rows x 16 columns)
static rs_status encode_maps(const rs_mesh *m, const double *psi, int ncol, sweep_maps &maps)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        RS_CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (!fn || qres != cudaDriverEntryPointSuccess) return rs_fail(RS_ERR_CUDA, "cuTensorMapEncodeTiled not available");
        encode = (encode_fn)fn;
    }
    static const cuuint32_t heights[SW_NBOX] = {1, 2, 4, 8, 16, 24};
    const cuuint64_t dims[2] = {(cuuint64_t)ncol, (cuuint64_t)(m->np + 1)};
    const cuuint64_t strides[1] = {(cuuint64_t)ncol * 8};
    const cuuint32_t estr[2] = {1, 1};
    for (int b = 0; b < SW_NBOX; ++b) {
        const cuuint32_t box[2] = {(cuuint32_t)SW_C, heights[b]};
        const CUresult r = encode(&maps.box[b], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double *>(psi), dims, strides, box,
                                  estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return rs_fail(RS_ERR_CUDA, "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")");
    }
    return RS_OK;
}

// The six tensor maps of a psi buffer are encoded once per (pointer, row pitch) and kept in the handle (a caller's
// block loop alternates between a few buffers): a warm apply does no driver call besides the launch.
static rs_status cached_maps(rs_mesh *m, const double *psi, int ncol, const sweep_maps **out)
{
    for (rs_sweep_map_cache &e : m->map_cache)
        if (e.psi == psi && e.ncol == ncol) {
            *out = reinterpret_cast<const sweep_maps *>(e.bytes);
            return RS_OK;
        }
    static_assert(sizeof(sweep_maps) <= sizeof(rs_sweep_map_cache::bytes), "tensor-map cache entry");
    if (m->map_cache.size() >= 16) m->map_cache.erase(m->map_cache.begin());   // oldest first
    m->map_cache.emplace_back();
    rs_sweep_map_cache &e = m->map_cache.back();
    e.psi = psi, e.ncol = ncol;
    const rs_status rc = encode_maps(m, psi, ncol, *reinterpret_cast<sweep_maps *>(e.bytes));
    if (rc != RS_OK) {
        m->map_cache.pop_back();
        return rc;
    }
    *out = reinterpret_cast<const sweep_maps *>(e.bytes);
    return RS_OK;
}

// measure = true (rs_hamiltonian_autotune only): every CTA also records its clock at the end of every step.
static rs_status launch_sweep(rs_mesh *m, int n, const rs_weights &w, const double *vloc, const double *psi, double *hpsi,
                              int ncol, cudaStream_t st, bool measure)
{
    if (!rs_sweep_supported(m, n, ncol)) return rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep kernel cannot serve this call");
    const rs_sweep_tables *tb = nullptr;
    rs_status rc = get_tables(m, n, ncol, &tb);
    if (rc != RS_OK) return rc;
    if (!tb->ok) return rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep tables: a plane needs more copy runs than a record holds");
    sweep_args a;
    a.items = tb->d_items, a.recs = tb->d_recs;
    a.vloc = vloc, a.psi = psi, a.hpsi = hpsi, a.ncol = (uint32_t)ncol;
    a.cycles = measure ? tb->d_cycles : nullptr;
    a.step_clock = measure ? tb->d_step_clock : nullptr;
    static const sweep_maps no_maps = {};
    const sweep_maps *maps = &no_maps;
    const bool tensor = ncol != SW_C || m->opt.force_tensor;
    if (tensor) {
        rc = cached_maps(m, psi, ncol, &maps);
        if (rc != RS_OK) return rc;
    }
    const unsigned grid = (unsigned)tb->nitems;
    if (tb->variant == VARIANT_N6)
        launch_shape<shape_n6>(tensor, grid, st, a, w, *maps);
    else
        launch_shape<shape_n4>(tensor, grid, st, a, w, *maps);
    RS_CUDA_TRY(cudaGetLastError());
    return RS_OK;
}

rs_status rs_launch_sweep(const rs_mesh *cm, int n, const rs_weights &w, const double *vloc, const double *psi,
                          double *hpsi, int ncol, cudaStream_t st)
{
    return launch_sweep(const_cast<rs_mesh *>(cm), n, w, vloc, psi, hpsi, ncol, st, false);   // the handle owns lazily filled caches
}

// Build and upload the tables of (mesh, n, ncol) now (rs_hamiltonian_prepare): afterwards rs_launch_sweep allocates
// nothing and never synchronises.
rs_status rs_sweep_prepare(const rs_mesh *cm, int n, int ncol)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    if (!rs_sweep_supported(m, n, ncol)) return rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep kernel cannot serve this call");
    const rs_sweep_tables *tb = nullptr;
    rs_status rc = get_tables(m, n, ncol, &tb);
    if (rc != RS_OK) return rc;
    return tb->ok ? RS_OK : rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep tables: a plane needs more copy runs than a record holds");
}

// true when the sweep kernel will really serve (mesh, n, ncol): supported and its tables could be built
bool rs_sweep_usable(const rs_mesh *cm, int n, int ncol)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    if (!rs_sweep_supported(m, n, ncol) || !m->have_device) return false;
    const rs_sweep_tables *tb = nullptr;
    return get_tables(m, n, ncol, &tb) == RS_OK && tb->ok;
}

int64_t rs_sweep_table_bytes(const rs_mesh *cm, int n, int ncol)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    if (!rs_sweep_supported(m, n, ncol)) return 0;
    auto f = m->sweep.find(std::make_pair(n * 16 + sweep_variant(n), ncol));
    if (f != m->sweep.end()) return f->second.bytes;
    rs_sweep_host h;   // no device (or not built yet): count on the host
    if (!rs_sweep_build_host(m, n, ncol, clamp_planes(m->opt.planes), sweep_nctas(m), h)) return 0;
    return (int64_t)(h.items.size() * sizeof(int2) + h.recs.size());
}

const char *rs_sweep_variant_name(const rs_mesh *m, int n, int ncol)
{
    const bool tensor = ncol != SW_C || m->opt.force_tensor;
    switch (sweep_variant(n)) {
        case VARIANT_N6:
            if (ncol == SW_HALF) return "sweep[n6 c8-in-16 8x16 q2p4 persistent ws tma2d+tmem s3]";
            return tensor ? "sweep[n6 c16 8x16 q2p4 persistent ws tma2d+tmem s3]" : "sweep[n6 c16 8x16 q2p4 persistent ws tma1d+tmem s3]";
        default:
            if (ncol == SW_HALF) return "sweep[n4 c8-in-16 16x16 q4p4 persistent ws tma2d+tmem s3]";
            return tensor ? "sweep[n4 c16 16x16 q4p4 persistent ws tma2d+tmem s3]" : "sweep[n4 c16 16x16 q4p4 persistent ws tma1d+tmem s3]";
    }
}

void rs_sweep_free(rs_mesh *m)
{
    for (auto &kv : m->sweep) {
        rs_sweep_tables &t = kv.second;
        cudaFree(t.d_items), cudaFree(t.d_recs), cudaFree(t.d_cycles), cudaFree(t.d_step_clock);
    }
    m->sweep.clear();
    m->map_cache.clear();
}

// ---------------------------------------------------------------------------------------------
// host self-check: replay the records symbolically (mesh indices instead of values) exactly as the
// kernel consumes them and verify that every output point sees, arm by arm, the neighbours that the
// plain table of rs_mesh_get_index_map names (reading S15), and that every (point, column slice) is
// produced exactly once.  Returns an empty string on success, else the first discrepancy.
// ---------------------------------------------------------------------------------------------
std::string rs_sweep_selfcheck_host(const rs_mesh *m, int n, int ncol, int max_planes, int nctas, int64_t *stats)
{
    if (!rs_sweep_supported(m, n, ncol)) return "unsupported (ordering / order / width)";
    rs_sweep_host h;
    if (!rs_sweep_build_host(m, n, ncol, max_planes, nctas, h)) return "a plane needs more copy runs than a record holds";
    const shape_rt sh = variant_shape(sweep_variant(n));
    const int N = sh.N, TY = sh.TY, TZ = SW_TZ, WY = sh.WY, WZ = sh.WZ, NS = 6 * N;
    const int64_t np = m->np;
    std::vector<int32_t> map((size_t)np * NS);
    rs_build_index_map(m, n, map.data());
    auto arm = [&](int32_t ip, int axis, int k) -> int32_t {   // k != 0; returns -1 for the zero slot
        const int32_t v = map[(size_t)ip * NS + axis * 2 * N + 2 * (std::abs(k) - 1) + (k > 0 ? 0 : 1)];
        return v == np ? -1 : v;
    };
    const int nchunks = sweep_nchunks(ncol);
    std::vector<uint8_t> done((size_t)np * nchunks, 0);
    int64_t npieces = 0;
    auto fail = [&](int cta, int step, const char *what, int y, int z, int k) {
        return std::string(what) + " (cta " + std::to_string(cta) + ", step " + std::to_string(step) + ", y " + std::to_string(y) +
               ", z " + std::to_string(z) + ", k " + std::to_string(k) + ")";
    };
    const int32_t UNK = -2;
    for (int cta = 0; cta < nctas; ++cta) {
        npieces += (int64_t)h.pieces[cta].size();
        std::vector<int32_t> stage((size_t)SW_STAGES * WY * WZ, UNK);
        // per tile point: centre values seen at the last 4 steps and the outputs pending from them
        std::vector<int32_t> hist((size_t)TY * TZ * N, UNK), pend((size_t)TY * TZ * N, -1), pend_chunk((size_t)TY * TZ * N, 0);
        const int nsteps = h.items[cta].y;
        for (int t = 0; t < nsteps; ++t) {
            const unsigned char *rec = h.recs.data() + (size_t)(h.items[cta].x + t) * sh.rec_bytes;
            const uint2 *runs = reinterpret_cast<const uint2 *>(rec + SW_REC_RUNS);
            const uint32_t *fill = reinterpret_cast<const uint32_t *>(rec + SW_REC_FILL);
            const uint32_t *hdr = reinterpret_cast<const uint32_t *>(rec + SW_REC_HDR);
            const int32_t *cidx = reinterpret_cast<const int32_t *>(rec + SW_REC_CIDX);
            int32_t *sg = &stage[(size_t)(t % SW_STAGES) * WY * WZ];
            uint32_t tx1 = 0;
            for (int r = 0; r < SW_MAXRUN; ++r) {
                const uint32_t len = runs[r].y >> 16, slot = runs[r].y & 0xffffu;
                if (slot + len > (uint32_t)(WY * WZ)) return fail(cta, t, "run leaves the stage", 0, 0, r);
                for (uint32_t i = 0; i < len; ++i) sg[slot + i] = (int32_t)(runs[r].x + i);
                tx1 += len * SW_SLOT_BYTES;
            }
            if (tx1 != hdr[2]) return fail(cta, t, "byte count of the copy runs", 0, 0, 0);
            {   // the clear list must name exactly the set bits of the bitmap; "whole stage": every slot without data is cleared
                const uint32_t nf = (hdr[0] >> HDR_NFILL_SHIFT) & 0xffu;
                const uint16_t *flist = reinterpret_cast<const uint16_t *>(rec + SW_REC_FLIST);
                if (nf == HDR_NFILL_WHOLE) {
                    std::vector<char> data((size_t)WY * WZ, 0);
                    for (int r = 0; r < SW_MAXRUN; ++r)
                        for (uint32_t i = 0; i < (runs[r].y >> 16); ++i) data[(runs[r].y & 0xffffu) + i] = 1;
                    for (int sl = 0; sl < WY * WZ; ++sl)
                        if ((((fill[sl >> 5] >> (sl & 31)) & 1u) != 0) == (data[sl] != 0)) return fail(cta, t, "whole-stage clear: bitmap", 0, 0, sl);
                } else {
                    uint32_t nbits = 0;
                    for (int sl = 0; sl < WY * WZ; ++sl)
                        if ((fill[sl >> 5] >> (sl & 31)) & 1u) {
                            if (nbits >= nf || flist[nbits] != sl) return fail(cta, t, "clear list and bitmap differ", 0, 0, sl);
                            ++nbits;
                        }
                    if (nbits != nf) return fail(cta, t, "clear list count", 0, 0, (int)nbits);
                }
            }
            for (int r = 0; r < WY; ++r)
                for (int z = 0; z < WZ; ++z)
                    if ((fill[(r * WZ + z) >> 5] >> ((r * WZ + z) & 31)) & 1u) sg[r * WZ + z] = -1;
            const int chunk = (int)hdr[1] / SW_C;
            const int ph = t % N;
            for (int y = 0; y < TY; ++y)
                for (int z = 0; z < TZ; ++z) {
                    const int wq = (y / sh.PY) * 2 + z / 8;
                    const int mode = (int)((hdr[0] >> (2 * wq)) & 3u);
                    const int32_t ci = (hdr[0] & HDR_OUTPUT_PLANE) ? cidx[y * TZ + z] : -1;
                    int32_t *hp = &hist[(size_t)(y * TZ + z) * N], *pp = &pend[(size_t)(y * TZ + z) * N];
                    int32_t *pc = &pend_chunk[(size_t)(y * TZ + z) * N];
                    const int32_t ce = mode == MODE_EMPTY ? -1 : sg[(N + y) * WZ + N + z];
                    // forward half of the x arm of the outputs pending from the last 4 steps
                    for (int k = 1; k <= N; ++k) {
                        const int32_t o = pp[(ph + N - k) % N];
                        if (k < N ? o >= 0 : false)
                            if (arm(o, 0, k) != ce) return fail(cta, t, "forward x arm", y, z, k);
                    }
                    {   // the output of plane t - 4 completes now
                        const int32_t o = pp[ph];
                        if (o >= 0) {
                            if (arm(o, 0, N) != ce) return fail(cta, t, "forward x arm", y, z, N);
                            uint8_t &d = done[(size_t)o * nchunks + pc[ph]];
                            if (d) return fail(cta, t, "output produced twice", y, z, 0);
                            d = 1;
                        }
                    }
                    if (ci >= 0) {
                        if (mode != MODE_FULL) return fail(cta, t, "output point in a warp that skips the plane", y, z, 0);
                        if (ce != ci) return fail(cta, t, "centre value", y, z, 0);
                        for (int k = 1; k <= N; ++k) {
                            if (sg[(N + y) * WZ + N + z + k] != arm(ci, 2, k)) return fail(cta, t, "z arm", y, z, k);
                            if (sg[(N + y) * WZ + N + z - k] != arm(ci, 2, -k)) return fail(cta, t, "z arm", y, z, -k);
                            if (sg[(N + y + k) * WZ + N + z] != arm(ci, 1, k)) return fail(cta, t, "y arm", y, z, k);
                            if (sg[(N + y - k) * WZ + N + z] != arm(ci, 1, -k)) return fail(cta, t, "y arm", y, z, -k);
                            if (hp[(ph + N - k) % N] != arm(ci, 0, -k)) return fail(cta, t, "backward x arm", y, z, -k);
                        }
                    }
                    pp[ph] = ci;
                    pc[ph] = chunk;
                    hp[ph] = ce;
                }
        }
        for (size_t q = 0; q < pend.size(); ++q)
            if (pend[q] >= 0) return fail(cta, nsteps, "output still pending at the end of the CTA's steps", 0, 0, 0);
    }
    for (size_t q = 0; q < done.size(); ++q)
        if (!done[q]) return "mesh point " + std::to_string(q / nchunks) + " slice " + std::to_string(q % nchunks) + " is never produced";
    if (stats) {
        stats[0] = nctas, stats[1] = h.nrec, stats[2] = npieces;
        stats[3] = (int64_t)(h.cost_max * 1000), stats[4] = (int64_t)(h.cost_mean * 1000);
        stats[5] = (int64_t)(h.items.size() * sizeof(int2) + h.recs.size());
        int64_t nfill = 0, nruns = 0;
        for (int64_t r = 0; r < h.nrec; ++r) {
            const unsigned char *rec = h.recs.data() + (size_t)r * sh.rec_bytes;
            for (int q = 0; q < 18; ++q) nfill += __builtin_popcount(reinterpret_cast<const uint32_t *>(rec + SW_REC_FILL)[q]);
            for (int q = 0; q < SW_MAXRUN; ++q) nruns += (reinterpret_cast<const uint2 *>(rec + SW_REC_RUNS)[q].y >> 16) != 0;
        }
        stats[6] = nfill, stats[7] = nruns;
    }
    return std::string();
}

// per-CTA {clock ticks of the last launch, steps, pieces, modelled load x 1000, full warp-steps}; returns the number of CTAs
int64_t rs_sweep_read_stats(const rs_mesh *cm, int n, int ncol, int64_t *out, int64_t max_ctas)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    auto f = m->sweep.find(std::make_pair(n * 16 + sweep_variant(n), ncol));
    if (f == m->sweep.end() || !f->second.ok) return 0;
    const rs_sweep_tables &t = f->second;
    const int64_t nc = std::min<int64_t>(t.nitems, max_ctas);
    std::vector<long long> cyc(t.nitems + 2048);
    if (cudaMemcpy(cyc.data(), t.d_cycles, cyc.size() * sizeof(long long), cudaMemcpyDeviceToHost) != cudaSuccess) return 0;
    for (int64_t c = 0; c < nc; ++c) {
        out[5 * c] = cyc[c];
        for (int k = 0; k < 4; ++k) out[5 * c + 1 + k] = t.host_stats[4 * c + k];
    }
    return nc;
}

// ---------------------------------------------------------------------------------------------
// Measure, don't guess: run the kernel on the caller's buffers, read the clock every CTA recorded at the end
// of every step, and deal the work again with the measured cost of each (tile, plane) instead of the model.
// The per-CTA residual of the model is systematic (run-to-run correlation 0.95-0.97 on B200), so it can be
// measured once per mesh.  Synchronises `st`.
// ---------------------------------------------------------------------------------------------
rs_status rs_sweep_autotune(const rs_mesh *cm, int n, const rs_weights &w, const double *vloc, const double *psi, double *hpsi,
                            int ncol, cudaStream_t st)
{
    rs_mesh *m = const_cast<rs_mesh *>(cm);
    if (!rs_sweep_supported(m, n, ncol)) return RS_OK;   // the gather kernel serves this call: nothing to tune
    const auto key = std::make_pair(n * 16 + sweep_variant(n), ncol);
    m->sweep_pieces.erase(key);   // a refined dealing of an earlier call: this call deals afresh
    rs_sweep_costs costs;
    // The measured costs depend a little on what runs beside a step, so a re-deal is not always better than the one before:
    // every dealing's slowest CTA is measured, and the best dealing seen (possibly the modelled one) is the one kept.
    long long best_max = -1;
    bool best_is_model = true, cur_is_model = m->sweep_costs.find(key) == m->sweep_costs.end();
    rs_sweep_costs best_costs, cur_costs;
    if (!cur_is_model) cur_costs = m->sweep_costs[key];
    // drop the device tables: the next use builds them again (from the costs / pieces then in the handle)
    auto drop_tables = [&]() {
        auto f = m->sweep.find(key);
        if (f != m->sweep.end()) {
            rs_sweep_tables &t = f->second;
            cudaFree(t.d_items), cudaFree(t.d_recs), cudaFree(t.d_cycles), cudaFree(t.d_step_clock);
            m->sweep.erase(f);
        }
    };
    auto slowest_cta = [&](const rs_sweep_tables *tb, long long *out) -> rs_status {
        std::vector<long long> cyc((size_t)tb->nitems);
        RS_CUDA_TRY(cudaMemcpy(cyc.data(), tb->d_cycles, cyc.size() * sizeof(long long), cudaMemcpyDeviceToHost));
        *out = *std::max_element(cyc.begin(), cyc.end());
        return RS_OK;
    };
    for (int round = 0; round < (m->opt.tune_rounds < 1 ? 1 : m->opt.tune_rounds); ++round) {   // later rounds measure the re-dealt work and refine it
        const rs_sweep_tables *tb = nullptr;
        rs_status rc = get_tables(m, n, ncol, &tb);
        if (rc != RS_OK) return rc;
        if (!tb->ok) return RS_OK;
        for (int rep = 0; rep < 3; ++rep) {
            rc = launch_sweep(m, n, w, vloc, psi, hpsi, ncol, st, true);
            if (rc != RS_OK) return rc;
        }
        RS_CUDA_TRY(cudaStreamSynchronize(st));
        {
            long long mx = 0;
            rc = slowest_cta(tb, &mx);
            if (rc != RS_OK) return rc;
            if (best_max < 0 || mx < best_max) best_max = mx, best_is_model = cur_is_model, best_costs = cur_costs;
        }
        std::vector<long long> clk((size_t)tb->nrec + 1);
        RS_CUDA_TRY(cudaMemcpy(clk.data(), tb->d_step_clock, clk.size() * sizeof(long long), cudaMemcpyDeviceToHost));
        const shape_rt sh = variant_shape(tb->variant);
        const size_t cells = (size_t)((m->dims[1] + sh.TY - 1) / sh.TY) * ((m->dims[2] + SW_TZ - 1) / SW_TZ) * m->dims[0];
        std::vector<double> sum(cells, 0.0);
        std::vector<int> cnt(cells, 0);
        double halo_sum = 0.0, full_sum = 0.0;
        int64_t halo_n = 0, full_n = 0;
        for (const int2 &it : tb->host_items)
            for (int t = 1; t < it.y; ++t) {   // step 0 has no predecessor to difference against
                const double d = (double)(clk[(size_t)it.x + t] - clk[(size_t)it.x + t - 1]);
                const int32_t cell = tb->rec_cell[(size_t)it.x + t];
                if (d <= 0.0 || d > 1e7) continue;
                if (cell < 0) {
                    halo_sum += d, ++halo_n;
                } else if ((size_t)cell < cells) {
                    sum[cell] += d, ++cnt[cell];
                    full_sum += d, ++full_n;
                }
            }
        if (!full_n || !halo_n) return RS_OK;
        costs.full.assign(cells, 0.f);
        for (size_t q = 0; q < cells; ++q)
            if (cnt[q]) costs.full[q] = (float)(sum[q] / cnt[q]);
        costs.halo = halo_sum / halo_n;
        costs.unit = full_sum / full_n;
        m->sweep_costs[key] = costs;
        cur_costs = costs, cur_is_model = false;
        drop_tables();   // the next use builds them with the measured costs
    }
    // if an earlier dealing was faster than the last one, go back to it
    auto measure = [&](std::vector<long long> &cyc, const rs_sweep_tables **tbo) -> rs_status {   // per-CTA clocks, mean of 3 launches
        const rs_sweep_tables *tb = nullptr;
        rs_status rc = get_tables(m, n, ncol, &tb);
        if (rc != RS_OK) return rc;
        if (!tb->ok) return rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep tables");
        cyc.assign((size_t)tb->nitems, 0);
        std::vector<long long> one((size_t)tb->nitems);
        for (int rep = 0; rep < 4; ++rep) {   // the first launch warms the tables up; the mean of the other three is used
            rc = launch_sweep(m, n, w, vloc, psi, hpsi, ncol, st, true);
            if (rc != RS_OK) return rc;
            RS_CUDA_TRY(cudaStreamSynchronize(st));
            if (rep == 0) continue;
            RS_CUDA_TRY(cudaMemcpy(one.data(), tb->d_cycles, one.size() * sizeof(long long), cudaMemcpyDeviceToHost));
            for (size_t c = 0; c < one.size(); ++c) cyc[c] += one[c] / 3;
        }
        *tbo = tb;
        return RS_OK;
    };
    std::vector<long long> cyc;
    const rs_sweep_tables *tb = nullptr;
    rs_status rc = measure(cyc, &tb);
    if (rc != RS_OK) return rc;
    if (best_max >= 0 && *std::max_element(cyc.begin(), cyc.end()) > best_max) {
        if (best_is_model)
            m->sweep_costs.erase(key);
        else
            m->sweep_costs[key] = best_costs;
        drop_tables();
        rc = measure(cyc, &tb);
        if (rc != RS_OK) return rc;
    }
    // ---- refinement: for a FIXED dealing the CTAs' times repeat from launch to launch (the error of the cost prediction is
    //      systematic per dealing), so the dealing is now only nudged: where a tile column is split between two CTAs the
    //      split plane moves towards the slower one (no new work piece, no new halo steps), a diffusion over the graph of
    //      CTAs that share columns.  The best dealing seen (slowest CTA) is kept.  What is left afterwards is the launch-to-launch
    //      scatter of a CTA's time (measured: rms 1.3-2.2 %, single CTAs 5-11 % off in one launch), which no static dealing removes.
    {
        std::vector<std::vector<rs_sweep_piece>> pieces = tb->pieces, best_pieces = tb->pieces;
        long long best = *std::max_element(cyc.begin(), cyc.end());
        const int nct = (int)pieces.size();
        const int min_len = m->opt.min_split < 1 ? 1 : m->opt.min_split;
        for (int round = 0; round < 2 * (m->opt.tune_rounds < 1 ? 1 : m->opt.tune_rounds); ++round) {
            // mean clocks per step of every CTA, boundaries of split columns
            std::vector<double> T(nct), per_plane(nct, 2500.0);
            std::vector<int> deg(nct, 0);
            for (int c = 0; c < nct; ++c) {
                T[c] = (double)cyc[c];
                int steps = 0;
                for (const rs_sweep_piece &pc : pieces[c]) steps += pc.xb - pc.xa + 2 * n;
                if (steps > 0) per_plane[c] = T[c] / steps;
            }
            struct edge { int ca, ia, cb, ib; };   // piece ia of CTA ca ends where piece ib of CTA cb begins
            std::vector<edge> edges;
            for (int ca = 0; ca < nct; ++ca)
                for (int ia = 0; ia < (int)pieces[ca].size(); ++ia)
                    for (int cb = 0; cb < nct; ++cb) {
                        if (cb == ca) continue;
                        for (int ib = 0; ib < (int)pieces[cb].size(); ++ib) {
                            const rs_sweep_piece &pa = pieces[ca][ia], &pb = pieces[cb][ib];
                            if (pa.iy == pb.iy && pa.iz == pb.iz && pa.chunk == pb.chunk && pa.xb == pb.xa) edges.push_back({ca, ia, cb, ib}), ++deg[ca], ++deg[cb];
                        }
                    }
            if (edges.empty()) break;
            {   // close enough: the slowest CTA within 1.5 % of the mean
                double mean = 0.0;
                for (int c = 0; c < nct; ++c) mean += T[c] / nct;
                if (*std::max_element(T.begin(), T.end()) < 1.015 * mean) break;
            }
            bool moved = false;
            for (const edge &e : edges) {
                rs_sweep_piece &pa = pieces[e.ca][e.ia], &pb = pieces[e.cb][e.ib];
                const double dT = T[e.ca] - T[e.cb];                       // > 0: the lower piece's CTA is slower -> it gives planes away
                const double c_plane = 0.5 * (per_plane[e.ca] + per_plane[e.cb]);
                int d = (int)std::lround(0.7 * dT / c_plane / std::max(deg[e.ca], deg[e.cb]));
                d = std::max(-8, std::min(8, d));
                if (d > 0) d = std::min(d, pa.xb - pa.xa - min_len);          // pa shrinks
                if (d < 0) d = -std::min(-d, pb.xb - pb.xa - min_len);        // pb shrinks
                if (d == 0 || (d > 0 && pa.xb - pa.xa - d < min_len) || (d < 0 && pb.xb - pb.xa + d < min_len)) continue;
                pa.xb -= d;
                pb.xa -= d;
                moved = true;
            }
            if (!moved) break;
            m->sweep_pieces[key] = pieces;
            drop_tables();
            rc = measure(cyc, &tb);
            if (rc != RS_OK) return rc;
            const long long mx = *std::max_element(cyc.begin(), cyc.end());
            if (mx < best) best = mx, best_pieces = pieces;
        }
        if (m->sweep_pieces.count(key) && m->sweep_pieces[key] != best_pieces) {
            m->sweep_pieces[key] = best_pieces;
            drop_tables();
            rc = measure(cyc, &tb);   // the tables in use are the best ones; rs_sweep_stats describes them
            if (rc != RS_OK) return rc;
        }
    }
    return RS_OK;
}
