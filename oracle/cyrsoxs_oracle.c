/*
 * cyrsoxs_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU statement of the P-RSoXS forward
 * simulation of arXiv 2209.13121 (CyRSoXS), written from the paper
 * (/root/reference/PAPER.md, cited below as P:<line>) and from the readings
 * fixed in DESIGN.md section 3 ("Readings of the paper").  It is the oracle
 * the CUDA path is compared against.  It shares no code, header, table or
 * constant generator with paper_2209_13121_b200/; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may call it.
 *
 * Everything follows the paper's order, angle by angle (Algorithm 1):
 *   O0  per-energy constants           (Eq. 1; n = 1 - delta + i beta)
 *   O1  e = U (1,0,0) = (cos z, sin z, 0)
 *   O2  p = sum_j (N_rot^j : N_rot^j - I) e / 4pi                 (Eq. 2-5)
 *   O3  p~ = FFT(p)   (textbook radix-2; an O(N^2) DFT beside it) (Eq. 6)
 *   O4  X(q) = | k^2 (I - r r^T) p~ |^2 on the Ewald sphere       (Eq. 7-8)
 *   O5  rotate the detector image back by the E-field angle
 *   O6  average over the angles
 * A second driver ("linear mode") uses only the linearity of O2-O4 in e
 * (p_zeta = cos z p_x + sin z p_y) so the large configurations stay affordable;
 * tests pin it to definition mode.
 *
 * Geometry decisions (validity, node indices, bilinear cells) are taken in
 * IEEE double with every operation rounded on its own: build with
 * -ffp-contract=off and never with -ffast-math.
 *
 * Pins (tests/test_oracle_pins.py): brute-force DFT, Parseval, closed forms for
 * a uniform film, split-material invariance, linearity in e, the isotropic
 * zeta law, form-factor zeros, mirror symmetry, two-fold anisotropy sign, the
 * binary-film closed form via numpy.fft, 90-degree exactness, grating direction,
 * q_z plane wave.  No function here is "parity unpinned" except the two
 * conventions DESIGN.md lists (image orientation, 0 for never-valid pixels).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define ORC_PI 3.141592653589793
#define ORC_HC_EV_NM 1239.84197 /* lambda[nm] = 1239.84197 / E[eV] (north_star) */

enum { ORC_EWALD_NEAREST = 0, ORC_EWALD_TRILINEAR = 1 };

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ O0 -- */

/* k = 2 pi / lambda, lambda = 1239.84197 / E.  The paper only names k_in "the
 * wavenumber of the incident wave"; the relation is north_star's. */
double orc_wavenumber(double energy_eV)
{
    double lambda = ORC_HC_EV_NM / energy_eV;
    return (2.0 * ORC_PI) / lambda;
}

/* Per material: n_par = 1 - delta_par + i beta_par, n_perp likewise (P:81,
 * north_star), n_iso = (n_par + 2 n_perp)/3 = Trace(N)/3 (Eq. 2).
 *   a = n_perp^2 - 1,  b = n_par^2 - n_perp^2,  c = n_iso^2 - 1,
 * each formed as (n-1)(n+1) with n-1 = -delta + i beta, so that nothing of
 * size 1 cancels.  Outputs are interleaved (re, im) doubles, n_mat each. */
void orc_coefficients(int n_mat, const float *delta_par, const float *beta_par,
                      const float *delta_perp, const float *beta_perp,
                      double *a, double *b, double *c)
{
    for (int m = 0; m < n_mat; ++m) {
        cplx npar_m1 = -(double)delta_par[m] + I * (double)beta_par[m];
        cplx nperp_m1 = -(double)delta_perp[m] + I * (double)beta_perp[m];
        cplx niso_m1 = (npar_m1 + 2.0 * nperp_m1) / 3.0;
        cplx am = nperp_m1 * (nperp_m1 + 2.0);
        cplx bm = (npar_m1 - nperp_m1) * (npar_m1 + nperp_m1 + 2.0);
        cplx cm = niso_m1 * (niso_m1 + 2.0);
        a[2 * m] = creal(am); a[2 * m + 1] = cimag(am);
        b[2 * m] = creal(bm); b[2 * m + 1] = cimag(bm);
        c[2 * m] = creal(cm); c[2 * m + 1] = cimag(cm);
    }
}

/* ------------------------------------------------------------------ O2 -- */

/* Induced polarization, Eq. 2-5 in the reading DESIGN.md 3-A1/A3:
 *   p = (1/4pi) sum_m phi_m [ S_m ( a_m e + b_m (d_m . e) d_m ) + (1 - S_m) c_m e ],
 *   d_m = (cos psi sin theta, sin psi sin theta, cos theta).
 * phi[m] etc. are N float32 values (promoted to double on read); S, theta, psi
 * may be NULL for an isotropic material (S == 0).  p* are N complex doubles. */
void orc_polarization(int64_t n_vox, int n_mat,
                      const float *const *phi, const float *const *S,
                      const float *const *theta, const float *const *psi,
                      const double *a, const double *b, const double *c,
                      double ex, double ey, double ez,
                      cplx *px, cplx *py, cplx *pz)
{
    const double inv4pi = 1.0 / (4.0 * ORC_PI);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_vox; ++i) {
        cplx sx = 0.0, sy = 0.0, sz = 0.0;
        for (int m = 0; m < n_mat; ++m) {
            double f = (double)phi[m][i];
            double s = S[m] ? (double)S[m][i] : 0.0;
            cplx am = a[2 * m] + I * a[2 * m + 1];
            cplx bm = b[2 * m] + I * b[2 * m + 1];
            cplx cm = c[2 * m] + I * c[2 * m + 1];
            /* unaligned part: (1 - s) (n_iso^2 - 1) e */
            cplx iso = (1.0 - s) * cm;
            cplx tx = iso * ex, ty = iso * ey, tz = iso * ez;
            if (s != 0.0) {
                double th = theta[m] ? (double)theta[m][i] : 0.0;
                double ps = psi[m] ? (double)psi[m][i] : 0.0;
                double dx = cos(ps) * sin(th);
                double dy = sin(ps) * sin(th);
                double dz = cos(th);
                double de = dx * ex + dy * ey + dz * ez;
                /* aligned part: s ( (n_perp^2-1) e + (n_par^2-n_perp^2) (d.e) d ) */
                tx += s * (am * ex + bm * (de * dx));
                ty += s * (am * ey + bm * (de * dy));
                tz += s * (am * ez + bm * (de * dz));
            }
            sx += f * tx; sy += f * ty; sz += f * tz;
        }
        px[i] = sx * inv4pi; py[i] = sy * inv4pi; pz[i] = sz * inv4pi;
    }
}

/* ------------------------------------------------------------------ O3 -- */

/* Textbook in-place iterative radix-2 decimation-in-time FFT, forward sign
 * exp(-2 pi i j k / n), unnormalised.  tw[j] = exp(-2 pi i j / n), j < n/2. */
static void fft1d_radix2(cplx *x, int n, const cplx *tw)
{
    for (int i = 1, j = 0; i < n; ++i) {          /* bit reversal */
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int i = 0; i < n; i += len)
            for (int j = 0; j < half; ++j) {
                cplx w = tw[j * step];
                cplx u = x[i + j], v = x[i + j + half] * w;
                x[i + j] = u + v;
                x[i + j + half] = u - v;
            }
    }
}

static cplx *make_twiddles(int n)
{
    int h = n / 2 > 0 ? n / 2 : 1;
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)h);
    for (int j = 0; j < h; ++j) {
        double ang = -2.0 * ORC_PI * (double)j / (double)n;
        tw[j] = cos(ang) + I * sin(ang);
    }
    return tw;
}

static int is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

/* Eq. 6 along one axis written out as the definition, O(n^2), for a length that is not a
 * power of two (the paper uses Nz = 63; DESIGN.md 3-A14): X[k] = sum_j x[j] exp(-2 pi i
 * j k / n).  The phase index j k mod n is exact integer arithmetic; ph[t] = exp(-2 pi i t / n),
 * t < n, is the table of the n distinct phases (make_phases). */
static void dft1d_definition(cplx *x, int n, cplx *scratch, const cplx *ph)
{
    for (int k = 0; k < n; ++k) {
        cplx acc = 0.0;
        for (int j = 0; j < n; ++j) acc += x[j] * ph[((int64_t)j * k) % n];
        scratch[k] = acc;
    }
    memcpy(x, scratch, sizeof(cplx) * (size_t)n);
}

static cplx *make_phases(int n)
{
    cplx *ph = (cplx *)malloc(sizeof(cplx) * (size_t)(n > 0 ? n : 1));
    for (int t = 0; t < n; ++t) {
        double ang = -2.0 * ORC_PI * (double)t / (double)n;
        ph[t] = cos(ang) + I * sin(ang);
    }
    return ph;
}

/* one line of length n, in place: radix-2 FFT for a power of two, the definition otherwise */
static void line_transform(cplx *x, int n, const cplx *tw, const cplx *ph, cplx *scratch)
{
    if (is_pow2(n)) fft1d_radix2(x, n, tw);
    else dft1d_definition(x, n, scratch, ph);
}

/* 3-D FFT of f[z][y][x] (x fastest), in place: Eq. 6, forward, unnormalised, origin at
 * voxel 0.  Any lengths (DESIGN.md 3-A14): an axis whose length is a power of two takes the
 * radix-2 FFT, any other axis the definition of Eq. 6. */
int orc_fft3(int Nx, int Ny, int Nz, cplx *f)
{
    if (Nx < 1 || Ny < 1 || Nz < 1) return -1;
    const int64_t sxy = (int64_t)Nx * Ny;
    cplx *twx = make_twiddles(Nx), *twy = make_twiddles(Ny), *twz = make_twiddles(Nz);
    cplx *phx = is_pow2(Nx) ? NULL : make_phases(Nx), *phy = is_pow2(Ny) ? NULL : make_phases(Ny),
         *phz = is_pow2(Nz) ? NULL : make_phases(Nz);
    /* along x: contiguous rows */
    if (Nx > 1) {
#pragma omp parallel
        {
            cplx *scr = (cplx *)malloc(sizeof(cplx) * (size_t)Nx);
#pragma omp for schedule(static)
            for (int64_t r = 0; r < (int64_t)Ny * Nz; ++r)
                line_transform(f + r * Nx, Nx, twx, phx, scr);
            free(scr);
        }
    }
    /* along y */
    if (Ny > 1) {
#pragma omp parallel
        {
            cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)Ny * 2);
#pragma omp for schedule(static)
            for (int64_t r = 0; r < (int64_t)Nx * Nz; ++r) {
                int64_t z = r / Nx, x = r % Nx;
                cplx *base = f + z * sxy + x;
                for (int y = 0; y < Ny; ++y) buf[y] = base[(int64_t)y * Nx];
                line_transform(buf, Ny, twy, phy, buf + Ny);
                for (int y = 0; y < Ny; ++y) base[(int64_t)y * Nx] = buf[y];
            }
            free(buf);
        }
    }
    /* along z */
    if (Nz > 1) {
#pragma omp parallel
        {
            cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)Nz * 2);
#pragma omp for schedule(static)
            for (int64_t r = 0; r < sxy; ++r) {
                cplx *base = f + r;
                for (int z = 0; z < Nz; ++z) buf[z] = base[(int64_t)z * sxy];
                line_transform(buf, Nz, twz, phz, buf + Nz);
                for (int z = 0; z < Nz; ++z) base[(int64_t)z * sxy] = buf[z];
            }
            free(buf);
        }
    }
    free(twx); free(twy); free(twz); free(phx); free(phy); free(phz);
    return 0;
}

/* The definition of Eq. 6 written out, O(N^2): for cross-checking orc_fft3 on
 * tiny inputs.  Any sizes.  out must not alias in. */
void orc_dft3_naive(int Nx, int Ny, int Nz, const cplx *in, cplx *out)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int kz = 0; kz < Nz; ++kz)
        for (int ky = 0; ky < Ny; ++ky)
            for (int kx = 0; kx < Nx; ++kx) {
                cplx acc = 0.0;
                for (int z = 0; z < Nz; ++z)
                    for (int y = 0; y < Ny; ++y)
                        for (int x = 0; x < Nx; ++x) {
                            double ph = (double)((int64_t)kx * x % Nx) / Nx
                                      + (double)((int64_t)ky * y % Ny) / Ny
                                      + (double)((int64_t)kz * z % Nz) / Nz;
                            double ang = -2.0 * ORC_PI * ph;
                            acc += in[((int64_t)z * Ny + y) * Nx + x] * (cos(ang) + I * sin(ang));
                        }
                out[((int64_t)kz * Ny + ky) * Nx + kx] = acc;
            }
}

/* Direct evaluation of p~ at a list of bins: the sum of Eq. 6 written out for those
 * bins only, over the polarization field that orc_polarization (O2, the single statement of
 * Eq. 2-5 in this file) produces slab by slab: O(n_vox * n_bins).  Used to spot-check sizes
 * where a whole double-precision FFT is too big.
 * bins: n_bins x 3 ints (kx, ky, kz), any integers (taken mod N).
 * out:  n_bins x 3 complex (p~x, p~y, p~z). */
void orc_polarization_dft_bins(int Nx, int Ny, int Nz, int n_mat,
                               const float *const *phi, const float *const *S,
                               const float *const *theta, const float *const *psi,
                               const double *a, const double *b, const double *c,
                               double ex, double ey, double ez,
                               int n_bins, const int *bins, cplx *out)
{
    const int64_t n_vox = (int64_t)Nx * Ny * Nz;
    const int64_t chunk = n_vox < ((int64_t)1 << 22) ? n_vox : ((int64_t)1 << 22);
    cplx *px = (cplx *)malloc(sizeof(cplx) * (size_t)chunk), *py = (cplx *)malloc(sizeof(cplx) * (size_t)chunk),
         *pz = (cplx *)malloc(sizeof(cplx) * (size_t)chunk);
    const float **tab = (const float **)malloc(sizeof(float *) * 4 * (size_t)n_mat);
    for (int q = 0; q < 3 * n_bins; ++q) out[q] = 0.0;
    for (int64_t i0 = 0; i0 < n_vox; i0 += chunk) {
        const int64_t n = n_vox - i0 < chunk ? n_vox - i0 : chunk;
        for (int m = 0; m < n_mat; ++m) {
            tab[m] = phi[m] + i0;
            tab[n_mat + m] = S[m] ? S[m] + i0 : NULL;
            tab[2 * n_mat + m] = theta[m] ? theta[m] + i0 : NULL;
            tab[3 * n_mat + m] = psi[m] ? psi[m] + i0 : NULL;
        }
        orc_polarization(n, n_mat, tab, tab + n_mat, tab + 2 * n_mat, tab + 3 * n_mat, a, b, c, ex, ey, ez, px, py, pz);
#pragma omp parallel for schedule(static)
        for (int q = 0; q < n_bins; ++q) {
            int64_t kx = ((bins[3 * q] % Nx) + Nx) % Nx;
            int64_t ky = ((bins[3 * q + 1] % Ny) + Ny) % Ny;
            int64_t kz = ((bins[3 * q + 2] % Nz) + Nz) % Nz;
            cplx sx = 0.0, sy = 0.0, sz = 0.0;
            for (int64_t l = 0; l < n; ++l) {
                const int64_t i = i0 + l;
                int x = (int)(i % Nx), y = (int)((i / Nx) % Ny), z = (int)(i / ((int64_t)Nx * Ny));
                double ph = (double)(kx * x % Nx) / Nx + (double)(ky * y % Ny) / Ny
                          + (double)(kz * z % Nz) / Nz;
                double ang = -2.0 * ORC_PI * ph;
                cplx w = cos(ang) + I * sin(ang);
                sx += px[l] * w; sy += py[l] * w; sz += pz[l] * w;
            }
            out[3 * q] += sx; out[3 * q + 1] += sy; out[3 * q + 2] += sz;
        }
    }
    free(px); free(py); free(pz); free(tab);
}

/* ------------------------------------------------------------------ O4 -- */

/* Geometry of one detector pixel (DESIGN.md 3-A5, A8, A11, A13).
 *   m_x = ix - Nx/2, q_x = m_x dq_x, dq = 2 pi / (N voxel)        (A5)
 *   s2  = (k k - q_x q_x) - q_y q_y ; invalid if s2 < 0            (Eq. 8, "real q_z")
 *   q_z = sqrt(s2) - k  (k_in = (0,0,k), normal incidence)
 *   g   = q_z / dq_z
 *   Nz == 1   : one node k_z = 0, weight 1                         (A13)
 *   NEAREST   : n = floor(g + 0.5); invalid if n < -Nz/2
 *   TRILINEAR : lo = floor(g), t = g - lo; nodes (lo, 1-t), (lo+1, t); a node
 *               of weight exactly 0 is not read; invalid if lo < -Nz/2
 * Returns the number of nodes (0 = invalid).  r = k_out / k = (q_x, q_y, q_z+k)/k. */
static int pixel_geometry(int Nx, int Ny, int Nz, double voxel, double k, int mode,
                          int ix, int iy, int node[2], double weight[2], double r[3])
{
    double dqx = (2.0 * ORC_PI) / ((double)Nx * voxel);
    double dqy = (2.0 * ORC_PI) / ((double)Ny * voxel);
    double dqz = (2.0 * ORC_PI) / ((double)Nz * voxel);
    double qx = (double)(ix - Nx / 2) * dqx;
    double qy = (double)(iy - Ny / 2) * dqy;
    double s2 = (k * k - qx * qx) - qy * qy;
    if (s2 < 0.0) return 0;
    double root = sqrt(s2);
    double qz = root - k;
    r[0] = qx / k; r[1] = qy / k; r[2] = (qz + k) / k;
    if (Nz == 1) { node[0] = 0; weight[0] = 1.0; return 1; }
    double g = qz / dqz;
    if (mode == ORC_EWALD_NEAREST) {
        double n = floor(g + 0.5);
        if (n < (double)(-(Nz / 2))) return 0;
        node[0] = (int)n; weight[0] = 1.0;
        return 1;
    }
    double lo = floor(g);
    if (lo < (double)(-(Nz / 2))) return 0;
    double t = g - lo;
    int cnt = 0;
    if (1.0 - t > 0.0) { node[cnt] = (int)lo; weight[cnt] = 1.0 - t; ++cnt; }
    if (t > 0.0) { node[cnt] = (int)lo + 1; weight[cnt] = t; ++cnt; }
    return cnt;
}

/* X at one grid node for the pixel's on-shell direction r (Eq. 7):
 *   w = p~ - r (r . p~),  X = k^4 ( |w_x|^2 + |w_y|^2 + |w_z|^2 ). */
static double scatter_X(double k, const double r[3], cplx vx, cplx vy, cplx vz)
{
    cplx rv = r[0] * vx + r[1] * vy + r[2] * vz;
    cplx wx = vx - r[0] * rv, wy = vy - r[1] * rv, wz = vz - r[2] * rv;
    double k2 = k * k;
    return (k2 * k2) * (creal(wx) * creal(wx) + cimag(wx) * cimag(wx)
                      + creal(wy) * creal(wy) + cimag(wy) * cimag(wy)
                      + creal(wz) * creal(wz) + cimag(wz) * cimag(wz));
}

static int64_t bin_index(int Nx, int Ny, int Nz, int mx, int my, int mz)
{
    int bx = ((mx % Nx) + Nx) % Nx, by = ((my % Ny) + Ny) % Ny, bz = ((mz % Nz) + Nz) % Nz;
    return ((int64_t)bz * Ny + by) * Nx + bx;
}

/* Ewald projection of X (Eq. 7-8): the detector image of one
 * E-field angle.  Image pixel (iy, ix) <-> (q_x, q_y) = ((ix-Nx/2) dq_x,
 * (iy-Ny/2) dq_y); X (the intensity, not p~) is interpolated linearly between
 * the two k_z neighbours.  img: Ny*Nx doubles (0 where invalid);
 * valid: Ny*Nx bytes. */
void orc_ewald(int Nx, int Ny, int Nz, double voxel, double k, int mode,
               const cplx *Px, const cplx *Py, const cplx *Pz,
               double *img, uint8_t *valid)
{
#pragma omp parallel for schedule(static)
    for (int iy = 0; iy < Ny; ++iy)
        for (int ix = 0; ix < Nx; ++ix) {
            int node[2]; double wt[2], r[3];
            int nn = pixel_geometry(Nx, Ny, Nz, voxel, k, mode, ix, iy, node, wt, r);
            double acc = 0.0;
            for (int j = 0; j < nn; ++j) {
                int64_t b = bin_index(Nx, Ny, Nz, ix - Nx / 2, iy - Ny / 2, node[j]);
                acc += wt[j] * scatter_X(k, r, Px[b], Py[b], Pz[b]);
            }
            img[(int64_t)iy * Nx + ix] = acc;
            valid[(int64_t)iy * Nx + ix] = (uint8_t)(nn > 0);
        }
}

/* The three real images of linear mode (tests pin them to orc_ewald):
 *   I_xx = sum_nodes wt k^4 |A P^x|^2, I_yy likewise, I_xy = sum wt k^4 Re<A P^x, A P^y>,
 * A = I - r r^T, so that I_zeta = C^2 I_xx + S^2 I_yy + 2 C S I_xy. */
void orc_ewald_linear(int Nx, int Ny, int Nz, double voxel, double k, int mode,
                      const cplx *Pxx, const cplx *Pxy, const cplx *Pxz,   /* p~ for e = x */
                      const cplx *Pyx, const cplx *Pyy, const cplx *Pyz,   /* p~ for e = y */
                      double *Ixx, double *Iyy, double *Ixy, uint8_t *valid)
{
#pragma omp parallel for schedule(static)
    for (int iy = 0; iy < Ny; ++iy)
        for (int ix = 0; ix < Nx; ++ix) {
            int node[2]; double wt[2], r[3];
            int nn = pixel_geometry(Nx, Ny, Nz, voxel, k, mode, ix, iy, node, wt, r);
            double axx = 0.0, ayy = 0.0, axy = 0.0, k2 = k * k;
            for (int j = 0; j < nn; ++j) {
                int64_t b = bin_index(Nx, Ny, Nz, ix - Nx / 2, iy - Ny / 2, node[j]);
                cplx u[3] = { Pxx[b], Pxy[b], Pxz[b] }, v[3] = { Pyx[b], Pyy[b], Pyz[b] };
                cplx ru = r[0] * u[0] + r[1] * u[1] + r[2] * u[2];
                cplx rv = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
                double sxx = 0.0, syy = 0.0, sxy = 0.0;
                for (int d = 0; d < 3; ++d) {
                    cplx wu = u[d] - r[d] * ru, wv = v[d] - r[d] * rv;
                    sxx += creal(wu) * creal(wu) + cimag(wu) * cimag(wu);
                    syy += creal(wv) * creal(wv) + cimag(wv) * cimag(wv);
                    sxy += creal(wu) * creal(wv) + cimag(wu) * cimag(wv);
                }
                axx += wt[j] * (k2 * k2) * sxx;
                ayy += wt[j] * (k2 * k2) * syy;
                axy += wt[j] * (k2 * k2) * sxy;
            }
            int64_t p = (int64_t)iy * Nx + ix;
            Ixx[p] = axx; Iyy[p] = ayy; Ixy[p] = axy;
            valid[p] = (uint8_t)(nn > 0);
        }
}

/* Geometry only, for tests: node indices (or INT32_MIN), weights, validity. */
void orc_ewald_nodes(int Nx, int Ny, int Nz, double voxel, double k, int mode,
                     int32_t *node0, int32_t *node1, double *w0, double *w1, uint8_t *valid)
{
    for (int iy = 0; iy < Ny; ++iy)
        for (int ix = 0; ix < Nx; ++ix) {
            int node[2] = { 0, 0 }; double wt[2] = { 0, 0 }, r[3];
            int nn = pixel_geometry(Nx, Ny, Nz, voxel, k, mode, ix, iy, node, wt, r);
            int64_t p = (int64_t)iy * Nx + ix;
            node0[p] = nn > 0 ? node[0] : INT32_MIN; w0[p] = nn > 0 ? wt[0] : 0.0;
            node1[p] = nn > 1 ? node[1] : INT32_MIN; w1[p] = nn > 1 ? wt[1] : 0.0;
            valid[p] = (uint8_t)(nn > 0);
        }
}

/* ------------------------------------------------------------- O1, O5 -- */

/* zeta in degrees -> (C, S) = (cos, sin) of zeta * (pi/180); a component below
 * 1e-15 in magnitude is snapped to 0 so that multiples of 90 degrees are exact
 * (DESIGN.md 3-A9). */
void orc_angle_cs(double zeta_deg, double *C, double *S)
{
    double zr = zeta_deg * (ORC_PI / 180.0);
    double c = cos(zr), s = sin(zr);
    if (fabs(c) < 1e-15) c = 0.0;
    if (fabs(s) < 1e-15) s = 0.0;
    *C = c; *S = s;
}

/* E_Angle[start, increment, end]: zeta_n = start + n step,
 * n = 0 .. floor((end - start)/step + 1e-9); start == end -> one angle. */
int orc_num_angles(double start_deg, double step_deg, double end_deg)
{
    if (start_deg == end_deg) return 1;
    if (step_deg == 0.0) return -1;
    double n = floor((end_deg - start_deg) / step_deg + 1e-9);
    if (n < 0.0) return -1;
    return (int)n + 1;
}

/* Rotate one angle's detector image back by the E-field angle about q = 0 and
 * accumulate ("we rotate the detector coordinates at the last step to
 * average"; reading DESIGN.md 3-A9, A10).  For output pixel (iy', ix'):
 *   u = ix' - Nx/2, v = iy' - Ny/2, rho = dq_y/dq_x = Nx/Ny (cubic voxels)
 *   f_x = (C u - S (v rho)) + Nx/2,   f_y = (S (u/rho) + C v) + Ny/2
 * i.e. the source is q = R(+zeta) q' in physical q.  Bilinear cell
 * x0 = floor f_x, alpha = f_x - x0 (y likewise); neighbour x0+1 is needed iff
 * alpha > 0, y0+1 iff beta > 0.  The sample is valid iff every needed
 * neighbour lies inside the image and is valid; then sum += sum_nb w I,
 * cnt += 1. */
void orc_rotate_accumulate(int Nx, int Ny, const double *img, const uint8_t *valid,
                           double C, double S, double *sum, uint32_t *cnt)
{
    const double rho = (double)Nx / (double)Ny;
#pragma omp parallel for schedule(static)
    for (int iy = 0; iy < Ny; ++iy)
        for (int ix = 0; ix < Nx; ++ix) {
            double u = (double)(ix - Nx / 2), v = (double)(iy - Ny / 2);
            double fx = (C * u - S * (v * rho)) + (double)(Nx / 2);
            double fy = (S * (u / rho) + C * v) + (double)(Ny / 2);
            double x0 = floor(fx), y0 = floor(fy);
            double al = fx - x0, be = fy - y0;
            int nx = al > 0.0 ? 2 : 1, ny = be > 0.0 ? 2 : 1;
            if (x0 < 0.0 || y0 < 0.0 || x0 + (nx - 1) > (double)(Nx - 1) || y0 + (ny - 1) > (double)(Ny - 1))
                continue;
            int X0 = (int)x0, Y0 = (int)y0, ok = 1;
            double acc = 0.0;
            for (int jy = 0; jy < ny && ok; ++jy)
                for (int jx = 0; jx < nx; ++jx) {
                    int64_t p = (int64_t)(Y0 + jy) * Nx + (X0 + jx);
                    if (!valid[p]) { ok = 0; break; }
                    double w = (jx ? al : 1.0 - al) * (jy ? be : 1.0 - be);
                    acc += w * img[p];
                }
            if (!ok) continue;
            sum[(int64_t)iy * Nx + ix] += acc;
            cnt[(int64_t)iy * Nx + ix] += 1u;
        }
}

/* O6 (P:253-255 with DESIGN.md 3-A10): out = sum / cnt, 0 where cnt == 0. */
void orc_finalize_average(int64_t n_pix, const double *sum, const uint32_t *cnt, double *out)
{
    for (int64_t p = 0; p < n_pix; ++p) out[p] = cnt[p] ? sum[p] / (double)cnt[p] : 0.0;
}

/* ------------------------------------------------------------- drivers -- */

/* Algorithm 1, definition mode, one energy: for every angle
 * O1 -> O2 -> O3 -> O4 -> O5, then O6.  out: Ny*Nx doubles, cnt: Ny*Nx.
 * Returns 0, -1 on a bad size/angle spec, -2 on allocation failure. */
int orc_run_energy(int Nx, int Ny, int Nz, int n_mat, double voxel,
                   const float *const *phi, const float *const *S,
                   const float *const *theta, const float *const *psi,
                   double energy_eV, const float *delta_par, const float *beta_par,
                   const float *delta_perp, const float *beta_perp,
                   double start_deg, double step_deg, double end_deg, int mode,
                   double *out, uint32_t *cnt)
{
    const int64_t n_vox = (int64_t)Nx * Ny * Nz, n_pix = (int64_t)Nx * Ny;
    int n_ang = orc_num_angles(start_deg, step_deg, end_deg);
    if (n_ang < 1 || Nx < 1 || Ny < 1 || Nz < 1) return -1;
    double k = orc_wavenumber(energy_eV);
    double *a = malloc(sizeof(double) * 2 * n_mat), *b = malloc(sizeof(double) * 2 * n_mat),
           *c = malloc(sizeof(double) * 2 * n_mat);
    cplx *px = malloc(sizeof(cplx) * n_vox), *py = malloc(sizeof(cplx) * n_vox),
         *pz = malloc(sizeof(cplx) * n_vox);
    double *img = malloc(sizeof(double) * n_pix), *sum = calloc(n_pix, sizeof(double));
    uint8_t *valid = malloc(n_pix);
    int rc = 0;
    if (!a || !b || !c || !px || !py || !pz || !img || !sum || !valid) { rc = -2; goto done; }
    orc_coefficients(n_mat, delta_par, beta_par, delta_perp, beta_perp, a, b, c);
    memset(cnt, 0, sizeof(uint32_t) * n_pix);
    for (int n = 0; n < n_ang; ++n) {
        double C, Sn;
        orc_angle_cs(start_deg + (double)n * step_deg, &C, &Sn);
        orc_polarization(n_vox, n_mat, phi, S, theta, psi, a, b, c, C, Sn, 0.0, px, py, pz);
        orc_fft3(Nx, Ny, Nz, px); orc_fft3(Nx, Ny, Nz, py); orc_fft3(Nx, Ny, Nz, pz);
        orc_ewald(Nx, Ny, Nz, voxel, k, mode, px, py, pz, img, valid);
        orc_rotate_accumulate(Nx, Ny, img, valid, C, Sn, sum, cnt);
    }
    orc_finalize_average(n_pix, sum, cnt, out);
done:
    free(a); free(b); free(c); free(px); free(py); free(pz); free(img); free(sum); free(valid);
    return rc;
}

/* Linear mode, one energy: p~ for e = x and e = y only (p is linear in e,
 * Eq. 5), the three real images of orc_ewald_linear, then per angle
 * I_zeta = C^2 I_xx + S^2 I_yy + 2 C S I_xy, O5, O6.  Same outputs as
 * orc_run_energy up to rounding (pinned by tests); used where definition mode
 * would take hours.  The y-field transforms reuse the x-field buffers one
 * after another, so the peak footprint is 6 complex fields. */
int orc_run_energy_linear(int Nx, int Ny, int Nz, int n_mat, double voxel,
                          const float *const *phi, const float *const *S,
                          const float *const *theta, const float *const *psi,
                          double energy_eV, const float *delta_par, const float *beta_par,
                          const float *delta_perp, const float *beta_perp,
                          double start_deg, double step_deg, double end_deg, int mode,
                          double *out, uint32_t *cnt,
                          double *Ixx_out, double *Iyy_out, double *Ixy_out, uint8_t *valid_out)
{
    const int64_t n_vox = (int64_t)Nx * Ny * Nz, n_pix = (int64_t)Nx * Ny;
    int n_ang = orc_num_angles(start_deg, step_deg, end_deg);
    if (n_ang < 1 || Nx < 1 || Ny < 1 || Nz < 1) return -1;
    double k = orc_wavenumber(energy_eV);
    double *a = malloc(sizeof(double) * 2 * n_mat), *b = malloc(sizeof(double) * 2 * n_mat),
           *c = malloc(sizeof(double) * 2 * n_mat);
    cplx *P[6] = { 0 };
    for (int i = 0; i < 6; ++i) P[i] = malloc(sizeof(cplx) * n_vox);
    double *Ixx = malloc(sizeof(double) * n_pix), *Iyy = malloc(sizeof(double) * n_pix),
           *Ixy = malloc(sizeof(double) * n_pix), *img = malloc(sizeof(double) * n_pix),
           *sum = calloc(n_pix, sizeof(double));
    uint8_t *valid = malloc(n_pix);
    int rc = 0;
    if (!a || !b || !c || !P[0] || !P[1] || !P[2] || !P[3] || !P[4] || !P[5] || !Ixx || !Iyy || !Ixy
        || !img || !sum || !valid) { rc = -2; goto done; }
    orc_coefficients(n_mat, delta_par, beta_par, delta_perp, beta_perp, a, b, c);
    orc_polarization(n_vox, n_mat, phi, S, theta, psi, a, b, c, 1.0, 0.0, 0.0, P[0], P[1], P[2]);
    orc_polarization(n_vox, n_mat, phi, S, theta, psi, a, b, c, 0.0, 1.0, 0.0, P[3], P[4], P[5]);
    for (int i = 0; i < 6; ++i) orc_fft3(Nx, Ny, Nz, P[i]);
    orc_ewald_linear(Nx, Ny, Nz, voxel, k, mode, P[0], P[1], P[2], P[3], P[4], P[5], Ixx, Iyy, Ixy, valid);
    memset(cnt, 0, sizeof(uint32_t) * n_pix);
    for (int n = 0; n < n_ang; ++n) {
        double C, Sn;
        orc_angle_cs(start_deg + (double)n * step_deg, &C, &Sn);
        for (int64_t p = 0; p < n_pix; ++p)
            img[p] = (C * C) * Ixx[p] + (Sn * Sn) * Iyy[p] + (2.0 * C * Sn) * Ixy[p];
        orc_rotate_accumulate(Nx, Ny, img, valid, C, Sn, sum, cnt);
    }
    orc_finalize_average(n_pix, sum, cnt, out);
    if (Ixx_out) memcpy(Ixx_out, Ixx, sizeof(double) * n_pix);
    if (Iyy_out) memcpy(Iyy_out, Iyy, sizeof(double) * n_pix);
    if (Ixy_out) memcpy(Ixy_out, Ixy, sizeof(double) * n_pix);
    if (valid_out) memcpy(valid_out, valid, n_pix);
done:
    free(a); free(b); free(c);
    for (int i = 0; i < 6; ++i) free(P[i]);
    free(Ixx); free(Iyy); free(Ixy); free(img); free(sum); free(valid);
    return rc;
}

/* ------------------------------------------------------- NEXT-1 reductions -- */

/* 1-D reductions of one detector image: the paper's
 * validation figures are expressed in the azimuthally averaged I(|q|) (Fig. 5b,
 * 8b), the scattering anisotropy A(q, E) (Fig. 15) and the
 * integrated scattering intensity ISI(E) (Fig. 6, Eq. 10).  The paper
 * gives no binning rule; readings:
 *   pixel (iy, ix): u = ix - Nx/2, v = (iy - Ny/2) * rho, rho = Nx/Ny (so that
 *   |q| = dq_x sqrt(u^2 + v^2)); radial bin b = floor(sqrt(u^2+v^2) + 1/2), kept
 *   if b < n_bins; only pixels with cnt > 0 take part (cnt == NULL: all do).
 *   I(b)      = mean of the image over the bin's valid pixels (0 if none);
 *   "para" sector: |v| <= tan_w |u| (within w of the q_x axis, which is the
 *   E-field axis after the rotate-back step); "perp" sector: |u| <= tan_w |v|;
 *   the pixel q = 0 belongs to neither;
 *   A(b)      = (I_para - I_perp) / (I_para + I_perp) with the sector means,
 *               0 where a sector is empty or the denominator is 0;
 *   ISI       = dq_x dq_y * sum of the image over all valid pixels (the 2-D
 *               detector integral; every valid pixel, not only those binned).
 * Outputs: Iq[n_bins], A[n_bins], npix[n_bins] (valid pixels per bin), *isi. */
void orc_reductions(int Nx, int Ny, double voxel, const double *img, const uint32_t *cnt,
                    int n_bins, double tan_w, double *Iq, double *A, uint32_t *npix, double *isi)
{
    double *sp = calloc((size_t)n_bins, sizeof(double)), *sq = calloc((size_t)n_bins, sizeof(double));
    uint32_t *np_ = calloc((size_t)n_bins, sizeof(uint32_t)), *nq = calloc((size_t)n_bins, sizeof(uint32_t));
    const double rho = (double)Nx / (double)Ny;
    const double dqx = (2.0 * ORC_PI) / ((double)Nx * voxel), dqy = (2.0 * ORC_PI) / ((double)Ny * voxel);
    double total = 0.0;
    for (int b = 0; b < n_bins; ++b) { Iq[b] = 0.0; A[b] = 0.0; npix[b] = 0; }
    for (int iy = 0; iy < Ny; ++iy)
        for (int ix = 0; ix < Nx; ++ix) {
            const int64_t p = (int64_t)iy * Nx + ix;
            if (cnt && cnt[p] == 0) continue;
            const double val = img[p];
            total += val;
            const double u = (double)(ix - Nx / 2), v = (double)(iy - Ny / 2) * rho;
            const double r = sqrt(u * u + v * v);
            const double fb = floor(r + 0.5);
            if (fb >= (double)n_bins) continue;
            const int b = (int)fb;
            Iq[b] += val; npix[b] += 1;
            if (u == 0.0 && v == 0.0) continue;
            if (fabs(v) <= tan_w * fabs(u)) { sp[b] += val; np_[b] += 1; }
            if (fabs(u) <= tan_w * fabs(v)) { sq[b] += val; nq[b] += 1; }
        }
    for (int b = 0; b < n_bins; ++b) {
        if (npix[b]) Iq[b] /= (double)npix[b];
        if (np_[b] && nq[b]) {
            const double ip = sp[b] / (double)np_[b], iq = sq[b] / (double)nq[b];
            if (ip + iq != 0.0) A[b] = (ip - iq) / (ip + iq);
        }
    }
    *isi = total * dqx * dqy;
    free(sp); free(sq); free(np_); free(nq);
}
