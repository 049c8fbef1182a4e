/*
 * oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU statement of what
 * the hot path of arxiv:1306.2953 computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call this.  It shares no code,
 * header, table or helper with the CUDA library under paper_1306_2953_b200/.
 *
 * What it states (fp64 throughout, "double precision for all operations"):
 *
 *   mesh      Omega = { (i,j,k) in Z^3 : min_A |h(i,j,k) - R_A| <= R }          PAPER.md:53 (sec. II,
 *             "uniform grid whose shape is given by the union of spheres around each atom"),
 *             PAPER.md:354 (sec. XII, radius / spacing).  Readings S3, S4 of DESIGN.md: closed
 *             ball, lattice through the origin, psi = 0 outside Omega.
 *
 *   H psi     (H psi)(p) = -1/2 (Lap psi)(p) + V(p) psi(p)                          PAPER.md:41 (eq. 2)
 *             (Lap psi)(p) = 1/h^2 [ 3 c_0 psi(p) + sum_{m=1..n} c_m sum_{axes} (psi(p+m e_a) + psi(p-m e_a)) ]
 *             PAPER.md:127 (sec. V.A: "the value at each point is calculated as a linear combination
 *             of the neighboring-point values ... fourth-order ... stencil size of 25"),
 *             PAPER.md:157 (sec. V.B: "multiply each orbitals by this potential").
 *             Reading S1: c_m are the standard central weights of f'' with half-width n.
 *
 *   layout    blocked[ip*B + j] = states[j][ip]                                      PAPER.md:101, Fig. 4 (:107)
 *
 * Parity pins (tests/test_oracle_pins.py): rational moment identities, constants, polynomials,
 * leading truncation term, plane-wave symbol, Hermiticity, dense 6^3 brute force, delta response,
 * Table I grid size, Fig. 4 worked example.  Nothing here is "parity unpinned".
 *
 * No blocking, no fusion, no reordering: one orbital at a time, triple loop over the bounding
 * lattice, inner loop over the star arms, every access bounds- and mask-checked.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---------- S1: central finite-difference weights of the second derivative ---------------------
 * c_m = 2 (-1)^(m+1) (n!)^2 / ( m^2 (n-m)! (n+m)! ),  m = 1..n;   c_0 = -2 sum_m c_m.
 * (n = 4: -205/72, 8/5, -1/5, 8/315, -1/560.)  Returns 0 on success.                           */
int orc_fd_coeffs(int n, double *c)
{
    if (n < 1 || n > 12 || !c) return 1;
    double sum = 0.0;
    for (int m = 1; m <= n; ++m) {
        /* (n!)^2 / ((n-m)! (n+m)!) = prod_{t=1..m} (n-m+t)/(n+t) */
        double r = 1.0;
        for (int t = 1; t <= m; ++t) r *= (double)(n - m + t) / (double)(n + t);
        double sign = (m % 2 == 1) ? 1.0 : -1.0;
        c[m] = 2.0 * sign * r / ((double)m * (double)m);
        sum += c[m];
    }
    c[0] = -2.0 * sum;
    return 0;
}

/* ---------- mesh: bounding lattice and in-domain mask ------------------------------------------ */
void orc_bbox(const double *centers, int nc, double R, double h, int lo[3], int dims[3])
{
    for (int a = 0; a < 3; ++a) {
        double mn = centers[a], mx = centers[a];
        for (int A = 1; A < nc; ++A) {
            double v = centers[3 * A + a];
            if (v < mn) mn = v;
            if (v > mx) mx = v;
        }
        int l = (int)floor((mn - R) / h) - 1;
        int u = (int)ceil((mx + R) / h) + 1;
        lo[a] = l;
        dims[a] = u - l + 1;
    }
}

/* mask[(ix*ny + iy)*nz + iz] = 1 iff lattice point (lo+ix, lo+iy, lo+iz)*h lies in the closed
 * ball of radius R around some centre.  Returns the number of in-domain points.               */
int64_t orc_mask(const double *centers, int nc, double R, double h, const int lo[3], const int dims[3],
                 uint8_t *mask)
{
    int64_t count = 0;
    const double R2 = R * R;
    for (int ix = 0; ix < dims[0]; ++ix)
        for (int iy = 0; iy < dims[1]; ++iy)
            for (int iz = 0; iz < dims[2]; ++iz) {
                const double x = (double)(lo[0] + ix) * h;
                const double y = (double)(lo[1] + iy) * h;
                const double z = (double)(lo[2] + iz) * h;
                uint8_t in = 0;
                for (int A = 0; A < nc && !in; ++A) {
                    const double dx = x - centers[3 * A + 0];
                    const double dy = y - centers[3 * A + 1];
                    const double dz = z - centers[3 * A + 2];
                    const double d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 <= R2) in = 1;
                }
                mask[((size_t)ix * dims[1] + iy) * dims[2] + iz] = in;
                count += in;
            }
    return count;
}

/* number of star arms (p, axis, +-m), p in Omega, m = 1..n, whose end point is outside Omega
 * (pin P11: must equal the number of zero-slot entries of the library's neighbour map).       */
int64_t orc_count_outside_arms(int n, const int dims[3], const uint8_t *mask)
{
    int64_t cnt = 0;
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    for (int ix = 0; ix < nx; ++ix)
        for (int iy = 0; iy < ny; ++iy)
            for (int iz = 0; iz < nz; ++iz) {
                if (!mask[((size_t)ix * ny + iy) * nz + iz]) continue;
                for (int m = -n; m <= n; ++m) {
                    if (m == 0) continue;
                    int jx = ix + m, jy = iy + m, jz = iz + m;
                    if (jx < 0 || jx >= nx || !mask[((size_t)jx * ny + iy) * nz + iz]) ++cnt;
                    if (jy < 0 || jy >= ny || !mask[((size_t)ix * ny + jy) * nz + iz]) ++cnt;
                    if (jz < 0 || jz >= nz || !mask[((size_t)ix * ny + iy) * nz + jz]) ++cnt;
                }
            }
    return cnt;
}

/* ---------- S5: the synthetic local potential (own code; the harness has its own copy) ---------
 * V(r) = sum_A -Z_A erf(rho_A / 0.5) / rho_A,  rho -> 0 limit -Z_A * 2/(0.5 sqrt(pi)).        */
void orc_vloc(const double *centers, const double *charges, int nc, const double *xyz, int64_t npts,
              double *v)
{
    const double soft = 0.5;
    const double lim = 2.0 / (soft * sqrt(acos(-1.0)));
    for (int64_t p = 0; p < npts; ++p) {
        double acc = 0.0;
        for (int A = 0; A < nc; ++A) {
            const double dx = xyz[3 * p + 0] - centers[3 * A + 0];
            const double dy = xyz[3 * p + 1] - centers[3 * A + 1];
            const double dz = xyz[3 * p + 2] - centers[3 * A + 2];
            const double rho = sqrt(dx * dx + dy * dy + dz * dz);
            acc -= charges[A] * (rho < 1e-12 ? lim : erf(rho / soft) / rho);
        }
        v[p] = acc;
    }
}

/* ---------- H psi on the dense bounding lattice ------------------------------------------------
 * psi, V, out: dense [nx][ny][nz] arrays (values at points outside Omega are ignored on input and
 * written as 0 on output).  periodic != 0 wraps every axis (test boxes; mask must be all ones).
 * `lanes` = 1 (real) or 2 (complex, interleaved re,im; V and the weights are real, so the two
 * lanes are two independent real problems -- PAPER.md:157, eq. 2).                              */
static inline double at(const double *f, const uint8_t *mask, const int dims[3], int periodic, int lanes,
                        int lane, int ix, int iy, int iz)
{
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    if (periodic) {
        ix = ((ix % nx) + nx) % nx;
        iy = ((iy % ny) + ny) % ny;
        iz = ((iz % nz) + nz) % nz;
    } else if (ix < 0 || ix >= nx || iy < 0 || iy >= ny || iz < 0 || iz >= nz) {
        return 0.0; /* S3: zero Dirichlet outside */
    }
    const size_t q = ((size_t)ix * ny + iy) * nz + iz;
    if (!mask[q]) return 0.0;
    return f[q * lanes + lane];
}

void orc_hpsi_dense(int n, const double *c, double h, const int dims[3], int periodic, const uint8_t *mask,
                    const double *V, const double *psi, double *out, int lanes)
{
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    const double pref = -0.5 / (h * h);
    for (int ix = 0; ix < nx; ++ix)
        for (int iy = 0; iy < ny; ++iy)
            for (int iz = 0; iz < nz; ++iz) {
                const size_t q = ((size_t)ix * ny + iy) * nz + iz;
                for (int l = 0; l < lanes; ++l) {
                    if (!mask[q]) { out[q * lanes + l] = 0.0; continue; }
                    const double p0 = psi[q * lanes + l];
                    double acc = 3.0 * c[0] * p0;
                    for (int m = 1; m <= n; ++m) {
                        const double sx = at(psi, mask, dims, periodic, lanes, l, ix + m, iy, iz)
                                        + at(psi, mask, dims, periodic, lanes, l, ix - m, iy, iz);
                        const double sy = at(psi, mask, dims, periodic, lanes, l, ix, iy + m, iz)
                                        + at(psi, mask, dims, periodic, lanes, l, ix, iy - m, iz);
                        const double sz = at(psi, mask, dims, periodic, lanes, l, ix, iy, iz + m)
                                        + at(psi, mask, dims, periodic, lanes, l, ix, iy, iz - m);
                        acc += c[m] * (sx + sy + sz);
                    }
                    out[q * lanes + l] = pref * acc + V[q] * p0;
                }
            }
}

/* Convenience driver used by the harness and the CPU baseline: nst orbitals given in canonical
 * (lexicographic, in-domain only) order psi[ist][np*lanes]; each is scattered into a dense box,
 * passed through orc_hpsi_dense, and gathered back.  canon[ip] = dense index of canonical point
 * ip.  One orbital at a time; `nthreads` > 1 only distributes whole orbitals over OpenMP threads
 * (orbitals are independent).  scratch: caller-provided, nthreads * 2 * nbox * lanes
 * doubles.  Returns the number of threads used.                                                */
int orc_hpsi_states(int n, const double *c, double h, const int dims[3], int periodic, const uint8_t *mask,
                    const double *Vdense, const int64_t *canon, int64_t np, const double *psi, double *out,
                    int nst, int lanes, int nthreads, double *scratch)
{
    const size_t nbox = (size_t)dims[0] * dims[1] * dims[2];
    int used = 1;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
    used = nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 1)
#endif
    for (int ist = 0; ist < nst; ++ist) {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double *din = scratch + (size_t)tid * 2 * nbox * lanes;
        double *dout = din + nbox * lanes;
        memset(din, 0, nbox * lanes * sizeof(double));
        const double *src = psi + (size_t)ist * np * lanes;
        double *dst = out + (size_t)ist * np * lanes;
        for (int64_t ip = 0; ip < np; ++ip)
            for (int l = 0; l < lanes; ++l) din[canon[ip] * lanes + l] = src[ip * lanes + l];
        orc_hpsi_dense(n, c, h, dims, periodic, mask, Vdense, din, dout, lanes);
        for (int64_t ip = 0; ip < np; ++ip)
            for (int l = 0; l < lanes; ++l) dst[ip * lanes + l] = dout[canon[ip] * lanes + l];
    }
    return used;
}

/* ---------- blocked layout (Fig. 4 at :107) --------------------------------------
 * states: [nst][ld] (each orbital contiguous, Fig. 4a);  block: [nrows][B] with the orbital index
 * fastest (Fig. 4b): block[ip*B + j] = states[ist0 + j][ip].  Columns j >= nst_in_block and rows
 * ip >= np are written as zero (reading S13: padded block, zero slot).  `lanes` as above; a
 * complex element moves as one unit.                                                          */
void orc_block_pack(const double *states, int64_t ld, int ist0, int nst_in_block, int B, int64_t np,
                    int64_t nrows, double *block, int lanes)
{
    for (int64_t ip = 0; ip < nrows; ++ip)
        for (int j = 0; j < B; ++j)
            for (int l = 0; l < lanes; ++l) {
                double v = 0.0;
                if (ip < np && j < nst_in_block) v = states[((size_t)(ist0 + j) * ld + ip) * lanes + l];
                block[((size_t)ip * B + j) * lanes + l] = v;
            }
}

void orc_block_unpack(const double *block, int B, int nst_in_block, int64_t np, double *states, int64_t ld,
                      int ist0, int lanes)
{
    for (int64_t ip = 0; ip < np; ++ip)
        for (int j = 0; j < nst_in_block; ++j)
            for (int l = 0; l < lanes; ++l)
                states[((size_t)(ist0 + j) * ld + ip) * lanes + l] = block[((size_t)ip * B + j) * lanes + l];
}
