// C-ABI entry points: argument checks, weight formation, kernel dispatch, host-buffer sweep.
#include <cstring>
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
    return RS_OK;
}

static rs_kernel resolve_kernel(const rs_mesh *m, int n, int ncol, rs_kernel k)
{
    // below ~1 M outputs the persistent kernel's start-up (tables, pipeline fill: ~20 us) outweighs its streaming rate
    // (measured: config 0 x 16 columns, gather 0.028 ms vs sweep 0.051 ms; config 1 x 16, 0.055 vs 0.051)
    if (k == RS_KERNEL_AUTO)
        return (m->np * (int64_t)ncol >= (1 << 20) && rs_sweep_usable(m, n, ncol)) ? RS_KERNEL_SWEEP : RS_KERNEL_GATHER;
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

// Whole path on host buffers (a7): H2D, then per block pack -> apply -> unpack, then D2H.
extern "C" rs_status rs_hamiltonian_apply_states_host(const rs_mesh *m, int n, const double *coeffs,
                                                      const double *vloc_host, const void *states_host,
                                                      void *hstates_host, int64_t ld, int nst_total, int B,
                                                      rs_dtype dtype)
{
    if (!m || !coeffs || !vloc_host || !states_host || !hstates_host || ld < m->np || nst_total < 1 ||
        !pow2_in(B, 1, RS_MAX_BLOCK) || n < 1 || n > m->max_n || (dtype != RS_REAL64 && dtype != RS_COMPLEX128))
        return rs_fail(RS_ERR_INVALID_ARG, "rs_hamiltonian_apply_states_host: bad argument");
    if (!m->have_device) return rs_fail(RS_ERR_CUDA, "no CUDA device");
    const size_t esz = dtype == RS_COMPLEX128 ? 16 : 8;
    const size_t sbytes = (size_t)nst_total * ld * esz, bbytes = rs_block_bytes(m, B, dtype);
    // Three streams: upload of block k + 1, compute of block k and download of block k - 1 overlap (PCIe is full duplex);
    // two pairs of block buffers so that compute never waits for its own previous unpack to drain.
    void *d_states = nullptr, *d_out = nullptr, *d_psi[2] = {nullptr, nullptr}, *d_hpsi[2] = {nullptr, nullptr};
    double *d_v = nullptr;
    cudaStream_t s_in = nullptr, s_cmp = nullptr, s_out = nullptr;
    const int nblocks = (nst_total + B - 1) / B;
    std::vector<cudaEvent_t> ev_in(nblocks, nullptr), ev_cmp(nblocks, nullptr);
    rs_status rc = RS_OK;
    auto cleanup = [&]() {
        cudaFree(d_states), cudaFree(d_out), cudaFree(d_psi[0]), cudaFree(d_psi[1]), cudaFree(d_hpsi[0]), cudaFree(d_hpsi[1]), cudaFree(d_v);
        for (cudaEvent_t e : ev_in)
            if (e) cudaEventDestroy(e);
        for (cudaEvent_t e : ev_cmp)
            if (e) cudaEventDestroy(e);
        if (s_in) cudaStreamDestroy(s_in);
        if (s_cmp) cudaStreamDestroy(s_cmp);
        if (s_out) cudaStreamDestroy(s_out);
    };
#define TRY_OR_CLEAN(call)                                                                     \
    do {                                                                                       \
        cudaError_t _e = (call);                                                               \
        if (_e != cudaSuccess) {                                                               \
            cudaDeviceSynchronize();                                                           \
            cleanup();                                                                         \
            return rs_fail(RS_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(_e));   \
        }                                                                                      \
    } while (0)
    TRY_OR_CLEAN(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
    TRY_OR_CLEAN(cudaStreamCreateWithFlags(&s_cmp, cudaStreamNonBlocking));
    TRY_OR_CLEAN(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
    TRY_OR_CLEAN(cudaMalloc(&d_states, sbytes));
    TRY_OR_CLEAN(cudaMalloc(&d_out, sbytes));
    for (int q = 0; q < 2; ++q) {
        TRY_OR_CLEAN(cudaMalloc(&d_psi[q], bbytes));
        TRY_OR_CLEAN(cudaMalloc(&d_hpsi[q], bbytes));
    }
    TRY_OR_CLEAN(cudaMalloc(&d_v, (size_t)m->np * 8));
    TRY_OR_CLEAN(cudaMemcpyAsync(d_v, vloc_host, (size_t)m->np * 8, cudaMemcpyHostToDevice, s_in));
    for (int k = 0; k < nblocks; ++k) {
        const int ist0 = k * B, nb = nst_total - ist0 < B ? nst_total - ist0 : B;
        const size_t off = (size_t)ist0 * ld * esz, bytes = (size_t)nb * ld * esz;
        TRY_OR_CLEAN(cudaEventCreateWithFlags(&ev_in[k], cudaEventDisableTiming));
        TRY_OR_CLEAN(cudaEventCreateWithFlags(&ev_cmp[k], cudaEventDisableTiming));
        TRY_OR_CLEAN(cudaMemcpyAsync((char *)d_states + off, (const char *)states_host + off, bytes, cudaMemcpyHostToDevice, s_in));
        TRY_OR_CLEAN(cudaEventRecord(ev_in[k], s_in));
        TRY_OR_CLEAN(cudaStreamWaitEvent(s_cmp, ev_in[k], 0));
        rc = rs_block_pack(m, d_states, ld, ist0, nb, B, d_psi[k & 1], dtype, s_cmp);
        if (rc == RS_OK) rc = rs_hamiltonian_apply(m, n, coeffs, d_v, d_psi[k & 1], d_hpsi[k & 1], B, dtype, s_cmp);
        if (rc == RS_OK) rc = rs_block_unpack(m, d_hpsi[k & 1], B, nb, d_out, ld, ist0, dtype, s_cmp);
        if (rc != RS_OK) {
            cudaDeviceSynchronize();
            cleanup();
            return rc;
        }
        TRY_OR_CLEAN(cudaEventRecord(ev_cmp[k], s_cmp));
        TRY_OR_CLEAN(cudaStreamWaitEvent(s_out, ev_cmp[k], 0));
        TRY_OR_CLEAN(cudaMemcpyAsync((char *)hstates_host + off, (const char *)d_out + off, bytes, cudaMemcpyDeviceToHost, s_out));
    }
    TRY_OR_CLEAN(cudaStreamSynchronize(s_out));
    TRY_OR_CLEAN(cudaStreamSynchronize(s_cmp));
    TRY_OR_CLEAN(cudaStreamSynchronize(s_in));
    cleanup();
#undef TRY_OR_CLEAN
    return RS_OK;
}

void rs_sweep_set_max_planes(int v);
void rs_sweep_set_force_tensor(int v);
void rs_sweep_set_nctas(int v);
void rs_sweep_set_shape(int v);
void rs_sweep_set_tuned_planes(int v);
void rs_sweep_set_min_split(int v);
void rs_sweep_set_tune_rounds(int v);
std::string rs_sweep_selfcheck_host(const rs_mesh *m, int n, int ncol, int max_planes, int nctas, int64_t *stats);

extern "C" rs_status rs_set_tuning(const char *name, int value)
{
    if (name && std::strcmp(name, "sweep_planes") == 0) {
        rs_sweep_set_max_planes(value);
        return RS_OK;
    }
    if (name && std::strcmp(name, "sweep_tensor") == 0) {
        rs_sweep_set_force_tensor(value);
        return RS_OK;
    }
    if (name && std::strcmp(name, "sweep_planes_tuned") == 0) {
        rs_sweep_set_tuned_planes(value);
        return RS_OK;
    }
    if (name && std::strcmp(name, "sweep_min_split") == 0) {
        rs_sweep_set_min_split(value);
        return RS_OK;
    }
    if (name && std::strcmp(name, "sweep_tune_rounds") == 0) {
        rs_sweep_set_tune_rounds(value);
        return RS_OK;
    }
    if (name && std::strcmp(name, "sweep_shape") == 0) {
        rs_sweep_set_shape(value);
        return RS_OK;
    }
    if (name && std::strcmp(name, "sweep_ctas") == 0) {
        rs_sweep_set_nctas(value);
        return RS_OK;
    }
    return rs_fail(RS_ERR_INVALID_ARG, "rs_set_tuning: unknown knob");
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
