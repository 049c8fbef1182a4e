// C-ABI entry points: argument checks, weight formation, kernel dispatch, host-buffer sweep.
#include <cstring>
#include <new>
#include <vector>

#include "rs_internal.h"

static bool pow2_in(int v, int lo, int hi) { return v >= lo && v <= hi && (v & (v - 1)) == 0; }

extern "C" rs_status rs_block_pack(const rs_mesh *m, const void *states, int64_t ld, int ist0, int nst_in, int B,
                                   void *block, rs_dtype dtype, void *stream)
{
    if (!m || !states || !block || ld < m->np || ist0 < 0 || !pow2_in(B, 1, RS_MAX_BLOCK) || nst_in < 1 || nst_in > B ||
        (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_block_pack: bad argument");
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    return rs_launch_pack(m, states, ld, ist0, nst_in, B, block, dtype == RS_COMPLEX128 ? 2 : 1, (cudaStream_t)stream);
}

extern "C" rs_status rs_block_unpack(const rs_mesh *m, const void *block, int B, int nst_in, void *states, int64_t ld,
                                     int ist0, rs_dtype dtype, void *stream)
{
    if (!m || !states || !block || ld < m->np || ist0 < 0 || !pow2_in(B, 1, RS_MAX_BLOCK) || nst_in < 1 || nst_in > B ||
        (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_block_unpack: bad argument");
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    return rs_launch_unpack(m, block, B, nst_in, states, ld, ist0, dtype == RS_COMPLEX128 ? 2 : 1, (cudaStream_t)stream);
}

static rs_status check_apply(const rs_mesh *m, int n, const double *coeffs, const double *vloc, const void *psi,
                             const void *hpsi, int nst, rs_dtype dtype)
{
    if (!m || !coeffs || !vloc || !psi || !hpsi) return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply: null argument");
    if (n < 1 || n > m->max_n) return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply: fd_order outside 1..max_fd_order");
    if (!pow2_in(nst, 1, RS_MAX_BLOCK)) return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply: nst must be 1,2,4,...,64");
    if (dtype != RS_REAL64 && dtype != RS_COMPLEX128) return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply: bad dtype");
    const size_t bytes = rs_block_bytes(m, nst, dtype);
    const char *a = (const char *)psi, *b = (const char *)hpsi;
    if (a == b || (a < b + bytes && b < a + bytes))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply: psi and hpsi overlap");
    // bulk copies (cp.async.bulk, tensor maps) and the 16-byte vector accesses of the gather kernel
    if ((((uintptr_t)psi | (uintptr_t)hpsi) & 15u) != 0)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply: psi and hpsi must be 16-byte aligned");
    if (((uintptr_t)vloc & 7u) != 0) return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply: vloc must be 8-byte aligned");
    return RS_OK;
}

static rs_kernel resolve_kernel(const rs_mesh *m, int n, int ncol, rs_kernel k)
{
    // below ~1 M outputs the persistent kernel's start-up (tables, pipeline fill: ~20 us) outweighs its streaming rate
    // (measured: config 0 x 16 columns, gather 0.028 ms vs sweep 0.051 ms; config 1 x 16, 0.055 vs 0.051)
    // 8 columns run as half a 16-column slice (the plane-sweep kernel does the work of 16): worth it only on large meshes
    // (measured: config 1, 0.25 M points: gather 0.025 ms vs sweep 0.033-0.040; config 2, 1.96 M points: 0.148 vs 0.139-0.148;
    // config 4, 3.8 M points: 0.284 vs 0.234-0.256, fd_order 6: 0.430 vs 0.298-0.348)
    if (k == RS_KERNEL_AUTO) {
        const int64_t outputs = m->np * (int64_t)ncol, least = ncol < 16 ? ((int64_t)1 << 23) + ((int64_t)1 << 22) : ((int64_t)1 << 20);
        return (outputs >= least && rs_sweep_usable(m, n, ncol)) ? RS_KERNEL_SWEEP : RS_KERNEL_GATHER;
    }
    return k;
}

extern "C" rs_status rs_hamiltonian_apply_v(const rs_mesh *m, int n, const double *coeffs, const double *vloc,
                                            const void *psi, void *hpsi, int nst, rs_dtype dtype, void *stream,
                                            rs_kernel kernel)
{
    rs_status st = check_apply(m, n, coeffs, vloc, psi, hpsi, nst, dtype);
    if (st != RS_OK) return st;
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    rs_weights w;
    std::memset(&w, 0, sizeof(w));
    for (int k = 0; k <= n; ++k) w.w[k] = -0.5 * coeffs[k] / (m->h * m->h);
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);  // complex = 2 independent real columns
    const rs_kernel k = resolve_kernel(m, n, ncol, kernel);
    if (k == RS_KERNEL_SWEEP) {
        if (!rs_sweep_supported(m, n, ncol)) return rs_fail(RS_ERR_UNSUPPORTED, "plane-sweep kernel cannot serve this call");
        return rs_launch_sweep(m, n, w, vloc, (const double *)psi, (double *)hpsi, ncol, (cudaStream_t)stream);
    }
    if (k != RS_KERNEL_GATHER) return rs_fail(RS_ERR_INVALID_ARG, "unknown kernel id");
    const int32_t *d_map = nullptr;
    st = rs_mesh_device_map(m, n, &d_map);
    if (st != RS_OK) return st;
    return rs_launch_gather(m, n, w, d_map, vloc, (const double *)psi, (double *)hpsi, ncol, (cudaStream_t)stream);
}

// ---- f1: block operations between orbitals (sec. VIII) -----------------------------------------
static rs_status check_blocks(const rs_mesh *m, const void *a, const void *b, int nst, rs_dtype dtype, const char *who)
{
    if (!m || !a || !b || !pow2_in(nst, 1, RS_MAX_BLOCK) || (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, std::string(who) + ": bad argument");
    if ((((uintptr_t)a | (uintptr_t)b) & 15u) != 0) return rs_fail(RS_ERR_INVALID_ARG, std::string(who) + ": blocks must be 16-byte aligned");
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    return RS_OK;
}

extern "C" rs_status rs_block_dot(const rs_mesh *m, const void *a, const void *b, int nst, rs_dtype dtype, void *out_dev, void *stream)
{
    if (!out_dev) return rs_fail(RS_ERR_INVALID_ARG, "rs_block_dot: null output");
    rs_status st = check_blocks(m, a, b, nst, dtype, "rs_block_dot");
    if (st != RS_OK) return st;
    const int lanes = dtype == RS_COMPLEX128 ? 2 : 1;
    return rs_launch_block_reduce(m, (const double *)a, (const double *)b, nullptr, nst * lanes, lanes, 1, lanes == 2 ? 1 : 0,
                                  (double *)out_dev, (cudaStream_t)stream);
}

extern "C" rs_status rs_block_expectation(const rs_mesh *m, const void *psi, const void *hpsi, const double *eps_dev, int nst,
                                          rs_dtype dtype, double *out_dev, void *stream)
{
    if (!out_dev) return rs_fail(RS_ERR_INVALID_ARG, "rs_block_expectation: null output");
    rs_status st = check_blocks(m, psi, hpsi, nst, dtype, "rs_block_expectation");
    if (st != RS_OK) return st;
    const int lanes = dtype == RS_COMPLEX128 ? 2 : 1;
    return rs_launch_block_reduce(m, (const double *)psi, (const double *)hpsi, eps_dev, nst * lanes, lanes, 3, 0, out_dev,
                                  (cudaStream_t)stream);
}

extern "C" rs_status rs_block_axpy(const rs_mesh *m, const void *alpha_dev, const void *x, void *y, int nst, rs_dtype dtype, void *stream)
{
    if (!alpha_dev || x == y) return rs_fail(RS_ERR_INVALID_ARG, "rs_block_axpy: null alpha or x == y");
    rs_status st = check_blocks(m, x, y, nst, dtype, "rs_block_axpy");
    if (st != RS_OK) return st;
    const int lanes = dtype == RS_COMPLEX128 ? 2 : 1;
    return rs_launch_block_axpy(m, (const double *)alpha_dev, (const double *)x, (double *)y, nst * lanes, lanes, (cudaStream_t)stream);
}

extern "C" rs_status rs_block_copy(const rs_mesh *m, const void *src, void *dst, int nst, rs_dtype dtype, void *stream)
{
    rs_status st = check_blocks(m, src, dst, nst, dtype, "rs_block_copy");
    if (st != RS_OK) return st;
    RS_CUDA_TRY(cudaMemcpyAsync(dst, src, rs_block_bytes(m, nst, dtype), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return RS_OK;
}

// ---- f2: overlap / subspace matrices over blocks of points (eqs. 5 and 7) -----------------------
extern "C" rs_status rs_block_overlap(const rs_mesh *m, const void *a, const void *b, int nst, rs_dtype dtype, void *M_dev, void *stream)
{
    if (!M_dev) return rs_fail(RS_ERR_INVALID_ARG, "rs_block_overlap: null output");
    rs_status st = check_blocks(m, a, b, nst, dtype, "rs_block_overlap");
    if (st != RS_OK) return st;
    const int lanes = dtype == RS_COMPLEX128 ? 2 : 1;
    if (nst * lanes == 1)   // a single real column: the 1 x 1 matrix is the dot product
        return rs_launch_block_reduce(m, (const double *)a, (const double *)b, nullptr, 1, 1, 1, 0, (double *)M_dev, (cudaStream_t)stream);
    return rs_launch_overlap(m, (const double *)a, (const double *)b, nst * lanes, lanes, (double *)M_dev, (cudaStream_t)stream);
}

// H psi and, from the same call, the per-orbital sums an eigensolver step needs.  The gather kernel and (for now) the
// plane-sweep kernel form the sums in a second streaming kernel over psi and H psi (one extra read of both blocks).
extern "C" rs_status rs_hamiltonian_apply_ex(const rs_mesh *m, int n, const double *coeffs, const double *vloc, const void *psi,
                                             void *hpsi, int nst, rs_dtype dtype, void *stream, const double *eps_dev,
                                             double *sums_dev)
{
    if (!sums_dev) return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply_ex: null output");
    rs_status st = rs_hamiltonian_apply_v(m, n, coeffs, vloc, psi, hpsi, nst, dtype, stream, RS_KERNEL_AUTO);
    if (st != RS_OK) return st;
    return rs_block_expectation(m, psi, hpsi, eps_dev, nst, dtype, sums_dev, stream);
}

extern "C" rs_status rs_hamiltonian_autotune(const rs_mesh *m, int n, const double *coeffs, const double *vloc, const void *psi,
                                             void *hpsi, int nst, rs_dtype dtype, void *stream)
{
    rs_status st = check_apply(m, n, coeffs, vloc, psi, hpsi, nst, dtype);
    if (st != RS_OK) return st;
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    rs_weights w;
    std::memset(&w, 0, sizeof(w));
    for (int k = 0; k <= n; ++k) w.w[k] = -0.5 * coeffs[k] / (m->h * m->h);
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);
    if (!rs_sweep_usable(m, n, ncol))   // only the gather kernel can serve this call: nothing to tune, just apply
        return rs_hamiltonian_apply(m, n, coeffs, vloc, psi, hpsi, nst, dtype, stream);
    return rs_sweep_autotune(m, n, w, vloc, (const double *)psi, (double *)hpsi, ncol, (cudaStream_t)stream);
}

extern "C" rs_status rs_hamiltonian_apply(const rs_mesh *m, int n, const double *coeffs, const double *vloc,
                                          const void *psi, void *hpsi, int nst, rs_dtype dtype, void *stream)
{
    return rs_hamiltonian_apply_v(m, n, coeffs, vloc, psi, hpsi, nst, dtype, stream, RS_KERNEL_AUTO);
}

extern "C" const char *rs_kernel_name(const rs_mesh *m, int n, int nst, rs_dtype dtype, rs_kernel kernel)
{
    if (!m) return "none";
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);
    return resolve_kernel(m, n, ncol, kernel) == RS_KERNEL_SWEEP ? rs_sweep_variant_name(m, n, ncol) : "gather";
}

extern "C" int64_t rs_kernel_table_bytes(const rs_mesh *m, int n, int nst, rs_dtype dtype, rs_kernel kernel)
{
    if (!m) return 0;
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);
    if (resolve_kernel(m, n, ncol, kernel) == RS_KERNEL_SWEEP) return rs_sweep_table_bytes(m, n, ncol);
    return m->np * 6 * (int64_t)n * 4;
}

// ---------------------------------------------------------------------------------------------
// Block sweep on HOST buffers (a7): a streaming driver.  A workspace owns a ring of `nbuf` block-sized device
// windows (states slab in, block, H block, states slab out), three streams and the events that order them;
// block k uses window k mod nbuf: upload of block k + 1, compute of block k and download of block k - 1 overlap
// (PCIe is full duplex).  Nothing is allocated per call and the device never holds more than nbuf blocks, so an
// orbital set larger than the HBM streams through (BASELINE.json configs[4]; sec. IV: block size vs memory).
// ---------------------------------------------------------------------------------------------
struct rs_workspace {
    const rs_mesh *m = nullptr;
    int B = 0, nbuf = 0;
    rs_dtype dtype = RS_REAL64;
    int64_t ld = 0;
    size_t esz = 8, slab = 0, bbytes = 0;
    std::vector<void *> d_in, d_out, d_psi, d_hpsi;
    double *d_v = nullptr;
    cudaStream_t s_in = nullptr, s_cmp = nullptr, s_out = nullptr;
    std::vector<cudaEvent_t> ev_in, ev_cmp, ev_out;
    cudaEvent_t ev_v = nullptr;
};

extern "C" rs_status rs_workspace_destroy(rs_workspace *ws)
{
    if (!ws) return RS_OK;
    if (ws->s_in) cudaStreamSynchronize(ws->s_in);
    if (ws->s_cmp) cudaStreamSynchronize(ws->s_cmp);
    if (ws->s_out) cudaStreamSynchronize(ws->s_out);
    for (auto *v : {&ws->d_in, &ws->d_out, &ws->d_psi, &ws->d_hpsi})
        for (void *p : *v) cudaFree(p);
    cudaFree(ws->d_v);
    for (auto *v : {&ws->ev_in, &ws->ev_cmp, &ws->ev_out})
        for (cudaEvent_t e : *v)
            if (e) cudaEventDestroy(e);
    if (ws->ev_v) cudaEventDestroy(ws->ev_v);
    if (ws->s_in) cudaStreamDestroy(ws->s_in);
    if (ws->s_cmp) cudaStreamDestroy(ws->s_cmp);
    if (ws->s_out) cudaStreamDestroy(ws->s_out);
    delete ws;
    return RS_OK;
}

extern "C" rs_status rs_workspace_create(const rs_mesh *m, int B, rs_dtype dtype, int64_t ld, int nbuf, rs_workspace **out)
{
    if (!m || !out || !pow2_in(B, 1, RS_MAX_BLOCK) || (dtype != RS_REAL64 && dtype != RS_COMPLEX128) || ld < m->np || nbuf < 2 || nbuf > 8)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_workspace_create: bad argument");
    *out = nullptr;
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    rs_workspace *ws = new (std::nothrow) rs_workspace;
    if (!ws) return rs_fail(RS_ERR_ALLOC, "out of host memory");
    ws->m = m, ws->B = B, ws->nbuf = nbuf, ws->dtype = dtype, ws->ld = ld;
    ws->esz = dtype == RS_COMPLEX128 ? 16 : 8;
    ws->slab = (size_t)B * ld * ws->esz;
    ws->bbytes = rs_block_bytes(m, B, dtype);
#define WS_TRY(call)                                                                               \
    do {                                                                                           \
        cudaError_t _e = (call);                                                                   \
        if (_e != cudaSuccess) {                                                                   \
            rs_workspace_destroy(ws);                                                              \
            return rs_fail(_e == cudaErrorMemoryAllocation ? RS_ERR_ALLOC : RS_ERR_CUDA,           \
                           std::string(#call) + ": " + cudaGetErrorString(_e));                    \
        }                                                                                          \
    } while (0)
    WS_TRY(cudaStreamCreateWithFlags(&ws->s_in, cudaStreamNonBlocking));
    WS_TRY(cudaStreamCreateWithFlags(&ws->s_cmp, cudaStreamNonBlocking));
    WS_TRY(cudaStreamCreateWithFlags(&ws->s_out, cudaStreamNonBlocking));
    WS_TRY(cudaEventCreateWithFlags(&ws->ev_v, cudaEventDisableTiming));
    WS_TRY(cudaMalloc(&ws->d_v, (size_t)m->np * 8));
    for (int q = 0; q < nbuf; ++q) {
        void *p = nullptr;
        cudaEvent_t e = nullptr;
        WS_TRY(cudaMalloc(&p, ws->slab));
        ws->d_in.push_back(p);
        WS_TRY(cudaMalloc(&p, ws->slab));
        ws->d_out.push_back(p);
        WS_TRY(cudaMalloc(&p, ws->bbytes));
        ws->d_psi.push_back(p);
        WS_TRY(cudaMalloc(&p, ws->bbytes));
        ws->d_hpsi.push_back(p);
        WS_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ws->ev_in.push_back(e);
        WS_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ws->ev_cmp.push_back(e);
        WS_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ws->ev_out.push_back(e);
    }
#undef WS_TRY
    *out = ws;
    return RS_OK;
}

extern "C" size_t rs_workspace_bytes(const rs_workspace *ws)
{
    return ws ? (size_t)ws->nbuf * 2 * (ws->slab + ws->bbytes) + (size_t)ws->m->np * 8 : 0;
}

extern "C" rs_status rs_hamiltonian_apply_states_stream(rs_workspace *ws, int n, const double *coeffs, const double *vloc_host,
                                                        const void *states_host, void *hstates_host, int nst_total)
{
    if (!ws || !coeffs || !vloc_host || !states_host || !hstates_host || nst_total < 1 || n < 1 || n > ws->m->max_n)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply_states_stream: bad argument");
    const rs_mesh *m = ws->m;
    const int B = ws->B, nblocks = (nst_total + B - 1) / B;
    const size_t esz = ws->esz, row = (size_t)m->np * esz, pitch = (size_t)ws->ld * esz;
    rs_status rc = rs_hamiltonian_prepare(m, n, B, ws->dtype);   // tables now, not inside the block loop
    if (rc != RS_OK) return rc;
#define WS_TRY(call)                                                                               \
    do {                                                                                           \
        cudaError_t _e = (call);                                                                   \
        if (_e != cudaSuccess) {                                                                   \
            cudaDeviceSynchronize();                                                               \
            return rs_fail(RS_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(_e));       \
        }                                                                                          \
    } while (0)
    WS_TRY(cudaMemcpyAsync(ws->d_v, vloc_host, (size_t)m->np * 8, cudaMemcpyHostToDevice, ws->s_in));
    WS_TRY(cudaEventRecord(ws->ev_v, ws->s_in));
    WS_TRY(cudaStreamWaitEvent(ws->s_cmp, ws->ev_v, 0));
    for (int k = 0; k < nblocks; ++k) {
        const int w = k % ws->nbuf, ist0 = k * B, nb = nst_total - ist0 < B ? nst_total - ist0 : B;
        const char *src = (const char *)states_host + (size_t)ist0 * pitch;
        char *dst = (char *)hstates_host + (size_t)ist0 * pitch;
        // upload: the window's previous pack (block k - nbuf) must have read its slab
        if (k >= ws->nbuf) WS_TRY(cudaStreamWaitEvent(ws->s_in, ws->ev_cmp[w], 0));
        if (pitch == row)
            WS_TRY(cudaMemcpyAsync(ws->d_in[w], src, (size_t)nb * row, cudaMemcpyHostToDevice, ws->s_in));
        else   // padded leading dimension: only the np points of every orbital travel
            WS_TRY(cudaMemcpy2DAsync(ws->d_in[w], pitch, src, pitch, row, nb, cudaMemcpyHostToDevice, ws->s_in));
        WS_TRY(cudaEventRecord(ws->ev_in[w], ws->s_in));
        // compute: after the upload, and after the window's previous download (block k - nbuf) left d_out
        WS_TRY(cudaStreamWaitEvent(ws->s_cmp, ws->ev_in[w], 0));
        if (k >= ws->nbuf) WS_TRY(cudaStreamWaitEvent(ws->s_cmp, ws->ev_out[w], 0));
        rc = rs_block_pack(m, ws->d_in[w], ws->ld, 0, nb, B, ws->d_psi[w], ws->dtype, ws->s_cmp);
        if (rc == RS_OK) rc = rs_hamiltonian_apply(m, n, coeffs, ws->d_v, ws->d_psi[w], ws->d_hpsi[w], B, ws->dtype, ws->s_cmp);
        if (rc == RS_OK) rc = rs_block_unpack(m, ws->d_hpsi[w], B, nb, ws->d_out[w], ws->ld, 0, ws->dtype, ws->s_cmp);
        if (rc != RS_OK) {
            cudaDeviceSynchronize();
            return rc;
        }
        WS_TRY(cudaEventRecord(ws->ev_cmp[w], ws->s_cmp));
        // download: unpack never writes beyond np, so only [0, np) of every row goes back (the caller's padding is untouched)
        WS_TRY(cudaStreamWaitEvent(ws->s_out, ws->ev_cmp[w], 0));
        if (pitch == row)
            WS_TRY(cudaMemcpyAsync(dst, ws->d_out[w], (size_t)nb * row, cudaMemcpyDeviceToHost, ws->s_out));
        else
            WS_TRY(cudaMemcpy2DAsync(dst, pitch, ws->d_out[w], pitch, row, nb, cudaMemcpyDeviceToHost, ws->s_out));
        WS_TRY(cudaEventRecord(ws->ev_out[w], ws->s_out));
    }
    WS_TRY(cudaStreamSynchronize(ws->s_out));
    WS_TRY(cudaStreamSynchronize(ws->s_cmp));
    WS_TRY(cudaStreamSynchronize(ws->s_in));
#undef WS_TRY
    return RS_OK;
}

// Convenience form: a temporary 3-window workspace per call (allocation inside; use the workspace form in a loop).
extern "C" rs_status rs_hamiltonian_apply_states_host(const rs_mesh *m, int n, const double *coeffs,
                                                      const double *vloc_host, const void *states_host,
                                                      void *hstates_host, int64_t ld, int nst_total, int B,
                                                      rs_dtype dtype)
{
    if (!m || !coeffs || !vloc_host || !states_host || !hstates_host || ld < m->np || nst_total < 1 ||
        !pow2_in(B, 1, RS_MAX_BLOCK) || n < 1 || n > m->max_n || (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply_states_host: bad argument");
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    rs_workspace *ws = nullptr;
    rs_status rc = rs_workspace_create(m, B, dtype, ld, 3, &ws);
    if (rc != RS_OK) return rc;
    rc = rs_hamiltonian_apply_states_stream(ws, n, coeffs, vloc_host, states_host, hstates_host, nst_total);
    rs_workspace_destroy(ws);
    return rc;
}

std::string rs_sweep_selfcheck_host(const rs_mesh *m, int n, int ncol, int max_planes, int nctas, int64_t *stats);

extern "C" rs_status rs_sweep_options_default(rs_sweep_options *out)
{
    if (!out) return rs_fail(RS_ERR_INVALID_ARG, "rs_sweep_options_default: null argument");
    *out = rs_mesh().opt;
    return RS_OK;
}

extern "C" rs_status rs_mesh_set_sweep_options(rs_mesh *m, const rs_sweep_options *opt)
{
    if (!m || !opt || opt->planes < 1 || opt->planes_tuned < 1 || opt->ctas < 0 || opt->min_split < 1 || opt->tune_rounds < 1)
        return rs_fail(RS_ERR_INVALID_ARG, "rs_mesh_set_sweep_options: bad argument");
    if (m->have_device) {
        RS_CUDA_TRY(cudaDeviceSynchronize());   // no launch may still read the tables that are dropped
        rs_sweep_free(m);
    }
    m->sweep_costs.clear();
    m->sweep_pieces.clear();
    m->opt = *opt;
    return RS_OK;
}

extern "C" rs_status rs_hamiltonian_prepare(const rs_mesh *m, int n, int nst, rs_dtype dtype)
{
    if (!m || n < 1 || n > m->max_n || !pow2_in(nst, 1, RS_MAX_BLOCK) || (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_prepare: bad argument");
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);
    if (resolve_kernel(m, n, ncol, RS_KERNEL_AUTO) == RS_KERNEL_SWEEP) {
        double *scr = nullptr;
        rs_status s2 = rs_reduce_scratch(m, &scr);
        if (s2 == RS_OK) s2 = rs_overlap_scratch(m, &scr);
        return s2 != RS_OK ? s2 : rs_sweep_prepare(m, n, ncol);
    }
    double *scratch = nullptr;
    rs_status st = rs_reduce_scratch(m, &scratch);   // the block reductions' per-CTA partial sums
    if (st == RS_OK) st = rs_overlap_scratch(m, &scratch);
    if (st != RS_OK) return st;
    const int32_t *d_map = nullptr;
    return rs_mesh_device_map(m, n, &d_map);
}

int64_t rs_sweep_read_stats(const rs_mesh *cm, int n, int ncol, int64_t *out, int64_t max_ctas);
extern "C" int64_t rs_sweep_stats(const rs_mesh *m, int n, int nst, rs_dtype dtype, int64_t *out_host, int64_t max_ctas)
{
    if (!m || !out_host || max_ctas < 1) return 0;
    return rs_sweep_read_stats(m, n, nst * (dtype == RS_COMPLEX128 ? 2 : 1), out_host, max_ctas);
}

extern "C" rs_status rs_sweep_selfcheck(const rs_mesh *m, int n, int nst, rs_dtype dtype, int max_planes, int nctas,
                                        int64_t *stats_host)
{
    if (!m || nst < 1 || max_planes < 4 || nctas < 1 || (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_sweep_selfcheck: bad argument");
    const int ncol = nst * (dtype == RS_COMPLEX128 ? 2 : 1);
    const std::string msg = rs_sweep_selfcheck_host(m, n, ncol, max_planes, nctas, stats_host);
    if (msg.rfind("unsupported", 0) == 0) return rs_fail(RS_ERR_UNSUPPORTED, msg);
    if (!msg.empty()) return rs_fail(RS_ERR_INVALID_ARG, "plane-sweep records: " + msg);
    return RS_OK;
}
