/*
 * rs.h -- C ABI of librs: batched Kohn-Sham  H psi = -1/2 Lap psi + V_loc psi  on a real-space mesh,
 * applied to a BLOCK of orbitals at once (arxiv:1306.2953; citations are /root/reference/PAPER.md
 * line + section).  Hand-written CUDA for sm_100a behind plain pointers; no torch types here.
 *
 * The problem, as the paper states it
 *   - H = -1/2 Lap + v(r), applied as an operator, never stored (PAPER.md:41 eq. 2; :119 sec. V).
 *   - The mesh is a uniform lattice of spacing h restricted to the union of spheres of radius R
 *     around the atoms (PAPER.md:53 sec. II; :354 sec. XII).  psi = 0 outside (reading S3).
 *   - Lap is a high-order finite-difference star: half-width n ("order"), 6n+1 points; the
 *     paper's "fourth-order ... stencil size of 25" is n = 4 (sec. V.A).
 *   - Routines receive a GROUP of orbitals (sec. IV); the block is stored with the
 *     orbital index fastest: element (point ip, orbital j) at  ip*B + j  (Fig. 4 :107).
 *     The block size B is a run-time power of two.
 *   - All local potentials are pre-summed into one array (sec. V.B).
 *   - Neighbours are found through a table because the shape is arbitrary.
 *
 * Conventions
 *   - "host"/"dev" on every pointer says where the memory lives.  The caller owns every buffer it
 *     passes; the mesh handle owns its own host tables and device tables.
 *   - Mesh order: the library chooses the enumeration of the np in-domain points (z-rows in
 *     lexicographic order by default); rs_mesh_get_points() publishes it.  Every per-point array (vloc, states, block
 *     rows) is indexed by that order.
 *   - Block layout: [nrows][ldb] elements, nrows = np + 1, ldb = B.  Row np is the ZERO SLOT: pack
 *     writes zeros there, apply never writes it, and apply REQUIRES it to be zero in psi.  Columns
 *     j >= nst_in_block are zero after pack and are ignored by unpack.
 *   - dtype RS_REAL64: element = double.  RS_COMPLEX128: element = interleaved (re, im) doubles; the
 *     weights and V are real, so a complex block of width B is computed as 2B independent real columns.
 *   - rs_block_pack / rs_block_unpack / rs_hamiltonian_apply are asynchronous on `stream`
 *     (a cudaStream_t passed as void*; NULL = legacy default stream).  After
 *     rs_hamiltonian_prepare(mesh, fd_order, nst, dtype) they allocate nothing and never synchronise.
 *     Without it, the first apply of a given (fd_order, block width) prepares lazily (host table build, one
 *     synchronous cudaMalloc + copy, cached in the handle); blocks of 8 or more than 16 real columns also encode
 *     their tensor maps once per psi buffer address (host-only work, cached).
 *   - Alignment: vloc 8 bytes; states 8 (real) / 16 (complex) bytes; block buffers (psi, hpsi) 16 bytes
 *     (bulk copies and vector accesses) -> RS_ERR_INVALID_ARG otherwise.
 *   - A mesh handle is not thread-safe; the library keeps no global state.
 *   - Every function returns rs_status; nothing throws.  rs_last_error() gives thread-local text for
 *     the last non-OK status.  There is no CPU fallback: without a CUDA device the compute entry
 *     points return RS_ERR_CUDA.
 */
#ifndef RS_H
#define RS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rs_mesh rs_mesh; /* opaque */

typedef enum {
    RS_OK = 0,
    RS_ERR_INVALID_ARG = 1,
    RS_ERR_ALLOC = 2,
    RS_ERR_CUDA = 3,
    RS_ERR_UNSUPPORTED = 4
} rs_status;

typedef enum { RS_REAL64 = 0, RS_COMPLEX128 = 1 } rs_dtype;

/* Point enumeration (sec. V.A, Fig. 7: "enumerate the grid points based on a
 * sequence of small parallelepipedic grids").  Results do not depend on it beyond rounding order. */
typedef enum {
    RS_ORDER_BRICK = 0, /* the paper's 4x4x4 bricks, brick after brick (gather kernel only; ablation of Fig. 8) */
    RS_ORDER_LEX = 1,   /* lexicographic (i, j, k), k fastest (default; what the plane-sweep kernel streams)    */
    RS_ORDER_TILE = 2   /* 16 x 16 tiles of the (j, k) plane, each marched along i: a tile's points of one plane are
                           consecutive (gather kernel only; ordering study)                          */
} rs_ordering;

/* Kernel selection for rs_hamiltonian_apply_v (tests and ablations; results agree to rounding). */
typedef enum {
    RS_KERNEL_AUTO = 0,   /* best available for this mesh / order / width                         */
    RS_KERNEL_GATHER = 1, /* per-point neighbour table, one gathered load per star arm (any mesh) */
    RS_KERNEL_SWEEP = 2   /* plane-sweep kernel: smem-staged planes + register x-window (RS_ORDER_LEX,
                             non-periodic mesh, fd_order 4 or 6, 16 | 32 | 64 | 128 real columns)  */
} rs_kernel;

#define RS_MAX_FD_ORDER 8
#define RS_MAX_BLOCK 64

/* ---- mesh (host builder; steps a1-a3 of SURVEY.md section 8(a)) ---------------------------------
 * rs_mesh_create: enumerate the lattice points (i,j,k)*spacing, integer i,j,k, lying in the closed
 * ball of `radius` around any of the `nc` centres (host [nc][3], bohr); choose the enumeration; build
 * the tables; upload them.  max_fd_order bounds the fd_order later passed to apply (1..RS_MAX_FD_ORDER).
 * Works without a CUDA device (tables stay on the host; compute calls then fail with RS_ERR_CUDA).   */
rs_status rs_mesh_create(const double *centers_host, int nc, double radius, double spacing,
                         int max_fd_order, rs_mesh **out);
rs_status rs_mesh_create_ordered(const double *centers_host, int nc, double radius, double spacing,
                                 int max_fd_order, rs_ordering ordering, rs_mesh **out);
/* Full rectangular test mesh, lattice indices 0..n-1 per axis.  periodic = 1 wraps all three axes
 * (then no arm ever leaves the mesh), periodic = 0 is zero-Dirichlet like the sphere meshes.        */
rs_status rs_mesh_create_box(int nx, int ny, int nz, double spacing, int max_fd_order, int periodic,
                             rs_ordering ordering, rs_mesh **out);
rs_status rs_mesh_destroy(rs_mesh *mesh);

int64_t rs_mesh_npoints(const rs_mesh *mesh);           /* np; -1 if mesh is NULL                   */
double rs_mesh_spacing(const rs_mesh *mesh);
int64_t rs_mesh_nbricks(const rs_mesh *mesh);           /* number of non-empty 4x4x4 bricks (0 for LEX) */
/* ijk_host [np][3] int32: lattice indices of the points, in mesh order.                            */
rs_status rs_mesh_get_points(const rs_mesh *mesh, int32_t *ijk_host);
/* map_host [np][6*fd_order] int32: entry (ip, s) is the mesh index of the point at arm s of ip, or np
 * (the zero slot) if that point is outside the mesh.  Arm order: s = axis*2n + 2*(k-1) + (0 for +k,
 * 1 for -k), axis 0 = i, k = 1..n.  This is the table of PAPER.md:131 in its plain form; the sweep
 * kernel uses a compact form that expands to exactly this (reading S15).                           */
rs_status rs_mesh_get_index_map(const rs_mesh *mesh, int fd_order, int32_t *map_host);

/* Bytes of one block buffer: (np + 1) * block_size * (8 or 16).  0 on bad arguments.               */
size_t rs_block_bytes(const rs_mesh *mesh, int block_size, rs_dtype dtype);

/* ---- layout transforms (steps a4, a6; Fig. 4) ---------------------------------------
 * states (dev): [nst_total][ld] elements, orbital-major (Fig. 4a), ld >= np, points in mesh order.
 * pack:   block[ip*B + j] = states[(ist0 + j)*ld + ip]   for j < nst_in_block, ip < np;
 *         zero for j >= nst_in_block and for row np.
 * unpack: states[(ist0 + j)*ld + ip] = block[ip*B + j]   for j < nst_in_block, ip < np.
 * block_size must be a power of two in 1..RS_MAX_BLOCK, 1 <= nst_in_block <= block_size.           */
rs_status rs_block_pack(const rs_mesh *mesh, const void *states_dev, int64_t ld, int ist0, int nst_in_block,
                        int block_size, void *block_dev, rs_dtype dtype, void *stream);
rs_status rs_block_unpack(const rs_mesh *mesh, const void *block_dev, int block_size, int nst_in_block,
                          void *states_dev, int64_t ld, int ist0, rs_dtype dtype, void *stream);

/* ---- the fused stencil + local potential (step a5; eq. 2 :41) -------------
 *   hpsi[ip][j] = -1/(2 h^2) [ 3 c_0 psi[ip][j] + sum_{m=1..n} c_m sum_{axes} (psi[ip + m e][j] + psi[ip - m e][j]) ]
 *                 + vloc[ip] psi[ip][j],      ip < np, j < nst;   psi = 0 outside the mesh.
 * coeffs_host: c_0..c_n, dimensionless (the library forms w_k = -0.5 c_k / h^2 in fp64, reading S6).
 * vloc_dev: [np] doubles, mesh order.  psi_dev / hpsi_dev: block buffers of width nst (= the block
 * size B of this call: 1, 2, 4, ..., 64), distinct and non-overlapping.  Row np of hpsi is left as is.
 * Errors: NULL pointers, nst not a power of two in 1..64, fd_order < 1 or > max_fd_order, psi and hpsi
 * overlapping, psi / hpsi not 16-byte aligned, vloc not 8-byte aligned -> RS_ERR_INVALID_ARG; launch failure or
 * no device -> RS_ERR_CUDA.                                                                         */
rs_status rs_hamiltonian_apply(const rs_mesh *mesh, int fd_order, const double *coeffs_host,
                               const double *vloc_dev, const void *psi_dev, void *hpsi_dev, int nst,
                               rs_dtype dtype, void *stream);
/* Same, with an explicit kernel choice; RS_ERR_UNSUPPORTED if that kernel cannot serve this call.  */
rs_status rs_hamiltonian_apply_v(const rs_mesh *mesh, int fd_order, const double *coeffs_host,
                                 const double *vloc_dev, const void *psi_dev, void *hpsi_dev, int nst,
                                 rs_dtype dtype, void *stream, rs_kernel kernel);

/* ---- block operations between orbitals (sec. VIII: "copies, linear
 * combinations, and dot products ... using the block-of-orbitals approach"; residuals for RMM-DIIS) ---
 * a, b, x, y, psi, hpsi: dev block buffers of width nst (layout above, 16-byte aligned).  Sums run over the np mesh
 * points, plain (no h^3 factor, reading S11), with the conjugate on the LEFT argument.  Asynchronous on `stream`;
 * results are deterministic (per-CTA partial sums in a scratch array owned by the mesh, added in a fixed order), so
 * reductions on one mesh must not run concurrently on two streams.
 *   rs_block_dot:          out_dev[j] = sum_p conj(a[p][j]) b[p][j], j < nst  (nst doubles, or nst (re, im) pairs)
 *   rs_block_expectation:  out_dev[0][j] = Re <psi_j|hpsi_j>, out_dev[1][j] = |psi_j|^2,
 *                          out_dev[2][j] = |hpsi_j - eps_j psi_j|^2 (eps_dev: nst real doubles, NULL = all 0): 3*nst doubles
 *   rs_block_axpy:         y[p][j] += alpha[j] x[p][j]; alpha_dev: nst elements of the block's dtype
 *   rs_block_copy:         dst = src (whole block, zero slot included)                                              */
rs_status rs_block_dot(const rs_mesh *mesh, const void *a_dev, const void *b_dev, int nst, rs_dtype dtype, void *out_dev,
                       void *stream);
rs_status rs_block_expectation(const rs_mesh *mesh, const void *psi_dev, const void *hpsi_dev, const double *eps_dev, int nst,
                               rs_dtype dtype, double *out_dev, void *stream);
/* rs_block_expectation for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): same arguments, bit-identical results, but the per-CTA partial sums live in a file-scope device array of
 * the library (1.73 MiB, held by every GPU that loads the library until the process exits) instead of scratch that the
 * first rs_block_expectation on a mesh allocates.  The call allocates and frees nothing and never synchronises.
 * Limit: nst * (dtype == RS_COMPLEX128 ? 2 : 1) <= 64 real columns; wider blocks -> RS_ERR_INVALID_ARG with a message
 * that names the limit.  The mesh's device must be the current device.  The array is shared by EVERY call on that
 * device, whatever the mesh or stream: two calls that overlap on the GPU race (order them on one stream or with
 * events); it needs no clearing between calls.  The first call per device resolves the array's address
 * (cudaGetSymbolAddress, no allocation): make that call outside graph capture.                                    */
rs_status rs_block_expectation_static(const rs_mesh *mesh, const void *psi_dev, const void *hpsi_dev, const double *eps_dev,
                                      int nst, rs_dtype dtype, double *out_dev, void *stream);
rs_status rs_block_axpy(const rs_mesh *mesh, const void *alpha_dev, const void *x_dev, void *y_dev, int nst, rs_dtype dtype,
                        void *stream);
rs_status rs_block_copy(const rs_mesh *mesh, const void *src_dev, void *dst_dev, int nst, rs_dtype dtype, void *stream);
/* ---- overlap and subspace matrices over blocks of points (SURVEY.md 8(f) row 2; PAPER.md:203-215 eq. 5, :225-235 eq. 7)
 *   M_dev[j][k] = sum_p conj(a[p][j]) b[p][k],  j, k < nst  (row-major [nst][nst] elements of the blocks' dtype)
 * With b = a this is a block of the overlap matrix S (eq. 5); with b = H a (rs_hamiltonian_apply's output) a block of the
 * subspace Hamiltonian h (eq. 7).  The block layout (all orbital coefficients of a point contiguous) is the paper's
 * "block-of-points" array, so the rank-k update runs on the blocks as they are: a hand-written fp64 tensor-core
 * (DMMA) contraction, deterministic (per-CTA partial matrices added in a fixed order by a second kernel).  Both blocks
 * have width nst.  Same stream rule as the reductions above.                                                    */
rs_status rs_block_overlap(const rs_mesh *mesh, const void *a_dev, const void *b_dev, int nst, rs_dtype dtype, void *M_dev,
                           void *stream);
/* rs_hamiltonian_apply plus, from the same call, sums_dev = the three rows of rs_block_expectation(psi, H psi, eps):
 * what one eigensolver step needs per orbital (Rayleigh quotient numerator and denominator, residual norm).        */
rs_status rs_hamiltonian_apply_ex(const rs_mesh *mesh, int fd_order, const double *coeffs_host, const double *vloc_dev,
                                  const void *psi_dev, void *hpsi_dev, int nst, rs_dtype dtype, void *stream,
                                  const double *eps_dev, double *sums_dev);

/* ---- non-local potential (sec. V.C, eq. 4 at :181) -------------------------------
 *   hpsi[r][j] += sum_A sum_lm gamma^A_lm(r - R_A) * h^3 sum_{r' in sphere A} gamma^A_lm(r' - R_A) psi[r'][j]
 * in the paper's two parts: the projection integrals are computed and stored, then multiplied by
 * the projectors and added.  The paper parallelises part 2 over atoms and therefore groups the atoms into colours whose
 * spheres share no mesh point (Fig. 11); here part 2 is a gather over the union of the spheres (every covered mesh point
 * adds up the atoms that cover it and is written once), which needs no colours and one launch.  The colouring is still
 * computed and published (rs_nonlocal_ncolors / rs_nonlocal_get_colors) for callers that scatter by atom themselves.
 * The sphere of atom A is the closed ball |r - R_A| <= rc restricted to the mesh (it may be empty).
 * The projector VALUES are an input (pseudopotential data, real): after rs_nonlocal_create the caller reads each atom's
 * sphere points (rs_nonlocal_sphere_size / rs_nonlocal_get_sphere: mesh indices, ascending), samples its nlm projectors
 * there and hands them over with rs_nonlocal_set_projectors (host [npts_A][nlm]).  nlm <= 16 (l_max = 3).
 * rs_nonlocal_apply ACCUMULATES into hpsi (call it after rs_hamiltonian_apply); asynchronous on `stream`; the first
 * call uploads the tables (rs_nonlocal_prepare does that ahead of time); deterministic (fixed-order sums, no atomics).
 * psi_dev / hpsi_dev: blocks of the mesh, 16-byte aligned, distinct.  Three kernels per call, chained by programmatic
 * dependent launch inside the call; to the rest of the stream the call behaves like one kernel.
 * The handle keeps per-call scratch: one apply at a time per handle.  The mesh must outlive the handle.           */
typedef struct rs_nonlocal rs_nonlocal; /* opaque */
rs_status rs_nonlocal_create(const rs_mesh *mesh, const double *centers_host, int natoms, double rc, int nlm,
                             rs_nonlocal **out);
rs_status rs_nonlocal_destroy(rs_nonlocal *nl);
int64_t rs_nonlocal_sphere_size(const rs_nonlocal *nl, int atom);                          /* -1 on bad arguments */
rs_status rs_nonlocal_get_sphere(const rs_nonlocal *nl, int atom, int32_t *mesh_index_host);
rs_status rs_nonlocal_set_projectors(rs_nonlocal *nl, int atom, const double *gamma_host);
int rs_nonlocal_ncolors(const rs_nonlocal *nl);
rs_status rs_nonlocal_get_colors(const rs_nonlocal *nl, int32_t *color_host /*[natoms]*/);
rs_status rs_nonlocal_prepare(rs_nonlocal *nl);
rs_status rs_nonlocal_apply(rs_nonlocal *nl, const void *psi_dev, void *hpsi_dev, int nst, rs_dtype dtype, void *stream);

/* Once per (mesh, fd_order, nst, dtype), before the first apply: build and upload the neighbour structure the chosen
 * kernel needs (plain table for the gather kernel, per-plane records for the plane-sweep kernel).  May allocate and
 * synchronise; afterwards rs_hamiltonian_apply for these arguments allocates nothing and never synchronises
 * (SURVEY.md section 8(b) conventions).  Idempotent.                                                              */
rs_status rs_hamiltonian_prepare(const rs_mesh *mesh, int fd_order, int nst, rs_dtype dtype);

/* Optional, once per (mesh, fd_order, nst, dtype): "measure, don't guess".  Runs the kernel a few times on the
 * caller's buffers (arguments as rs_hamiltonian_apply; hpsi receives H psi), reads back the clock each persistent
 * CTA recorded at the end of every plane, and deals the work to the CTAs again using the measured cost of every
 * (tile, plane) instead of the built-in cost model, then refines that dealing by moving the planes at which a tile column is
 * split between two CTAs towards the slower one; the fastest dealing measured is kept (about 0.5-1 s once per mesh, order and
 * width).  Later rs_hamiltonian_apply calls use the re-dealt tables; results
 * are unchanged up to rounding order.  SYNCHRONISES `stream` and replaces the mesh's device tables: no other call
 * on this mesh may be in flight on another stream or thread.  A call that only the gather kernel can serve is just
 * applied.                                                                                                        */
rs_status rs_hamiltonian_autotune(const rs_mesh *mesh, int fd_order, const double *coeffs_host,
                                  const double *vloc_dev, const void *psi_dev, void *hpsi_dev, int nst,
                                  rs_dtype dtype, void *stream);

/* ---- whole path on HOST buffers (step a7: the block sweep; used for the end-to-end number) --------
 * A workspace owns a ring of `nbuf` (2..8; 3 = upload / compute / download all overlapped) block-sized device
 * windows, three streams and their events for blocks of `block_size` orbitals of `dtype` with leading dimension ld
 * (>= np).  Device memory held: nbuf * 2 * (block_size*ld*elem + rs_block_bytes) + 8 np  (rs_workspace_bytes);
 * it does not depend on the number of orbitals, so sets larger than the HBM stream through (BASELINE.json
 * configs[4]: 1024 orbitals "processed in blocks ... streamed through HBM"; sec. IV).
 * RS_ERR_ALLOC if the device memory cannot be had.                                                              */
typedef struct rs_workspace rs_workspace; /* opaque */
rs_status rs_workspace_create(const rs_mesh *mesh, int block_size, rs_dtype dtype, int64_t ld, int nbuf,
                              rs_workspace **out);
rs_status rs_workspace_destroy(rs_workspace *ws);
size_t rs_workspace_bytes(const rs_workspace *ws);
/* states_host / hstates_host: pinned (for overlap) or pageable host arrays [nst_total][ld], mesh order; vloc_host
 * [np].  For each block of block_size orbitals: upload, pack, apply, unpack, download -- one cudaMemcpyAsync per
 * block per direction, nothing allocated, pipelined over the ring.  Only the np points of every orbital are
 * written to hstates_host (padding columns ld > np keep the caller's contents).  Returns after the last
 * download has completed (synchronises its own three streams only).  The mesh must outlive the workspace.      */
rs_status rs_hamiltonian_apply_states_stream(rs_workspace *ws, int fd_order, const double *coeffs_host,
                                             const double *vloc_host, const void *states_host, void *hstates_host,
                                             int nst_total);
/* Convenience form of the same: creates a 3-window workspace, streams, destroys it (allocation per call).      */
rs_status rs_hamiltonian_apply_states_host(const rs_mesh *mesh, int fd_order, const double *coeffs_host,
                                           const double *vloc_host, const void *states_host,
                                           void *hstates_host, int64_t ld, int nst_total, int block_size,
                                           rs_dtype dtype);

const char *rs_last_error(void);
/* Static description of the kernel rs_hamiltonian_apply would pick ("gather", "sweep[...]").       */
const char *rs_kernel_name(const rs_mesh *mesh, int fd_order, int nst, rs_dtype dtype, rs_kernel kernel);
/* Bytes of neighbour structure the chosen kernel reads per call (for the roofline's algorithmic bytes). */
int64_t rs_kernel_table_bytes(const rs_mesh *mesh, int fd_order, int nst, rs_dtype dtype, rs_kernel kernel);
int rs_version(void);
/* Options of the plane-sweep kernel's host-side work dealing, PER MESH (no process-global state).  Defaults:
 * rs_sweep_options_default().  rs_mesh_set_sweep_options() drops the tables (and measured costs) built so far, so
 * the next prepare / apply builds them under the new options; it synchronises the device.  For tests and ablations;
 * normal use never needs it (the block size is the only run-time knob of the method).               */
typedef struct {
    int planes;        /* x-slab thickness of a work item while the step costs are modelled (default 32)            */
    int planes_tuned;  /* the same once rs_hamiltonian_autotune measured them (default 1 << 20: whole tile columns)  */
    int ctas;          /* persistent CTAs (0 = one per SM)                                                          */
    int force_tensor;  /* 1 = use the 2-D tensor-map copies also for 16-column blocks                               */
    int min_split;     /* fewest output planes of a work piece cut off when dealing (default 3)                     */
    int tune_rounds;   /* measure / re-deal rounds of rs_hamiltonian_autotune (default 3); it then runs up to twice as
                          many refinement rounds that only move the split planes of shared tile columns               */
} rs_sweep_options;
rs_status rs_sweep_options_default(rs_sweep_options *out);
rs_status rs_mesh_set_sweep_options(rs_mesh *mesh, const rs_sweep_options *opt);
/* Host-only diagnostic (no device needed): build the plane-sweep kernel's compact records for (mesh,
 * fd_order, block width nst of dtype) dealt to `nctas` CTAs with slabs of `max_planes`, replay them
 * symbolically and verify that they expand to exactly the plain table of rs_mesh_get_index_map and that
 * every (point, 16-column slice) is produced exactly once (reading S15 of DESIGN.md).  stats_host (may be
 * NULL) receives 8 values: {nctas, records, work pieces, modelled cost of the busiest CTA x1000, of the average
 * CTA x1000, table bytes, slots zero-filled over all records, copy runs over all records}.  RS_ERR_UNSUPPORTED if
 * the sweep kernel cannot serve the call; a discrepancy ->
 * RS_ERR_INVALID_ARG with the first offending (CTA, step, point, arm) in rs_last_error().               */
rs_status rs_sweep_selfcheck(const rs_mesh *mesh, int fd_order, int nst, rs_dtype dtype, int max_planes, int nctas,
                             int64_t *stats_host);

/* Per-CTA figures of the plane-sweep kernel's last launch for (mesh, fd_order, nst, dtype), for calibrating
 * the cost model that deals work to the persistent CTAs: out_host [max_ctas][5] = {clock ticks spent in the last
 * MEASURING launch (rs_hamiltonian_autotune; production launches record nothing), steps, work pieces, modelled
 * load x1000, full warp-steps}.  Synchronises the device.  Returns the number of CTAs written (0 if no tables).  */
int64_t rs_sweep_stats(const rs_mesh *mesh, int fd_order, int nst, rs_dtype dtype, int64_t *out_host, int64_t max_ctas);

#ifdef __cplusplus
}
#endif
#endif /* RS_H */
