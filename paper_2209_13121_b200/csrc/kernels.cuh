// kernels.cuh -- the sm_100a kernels of the CyRSoXS hot path.
//   k_xpass_chi   polarization (Eq. 2-5) fused with the FFT along x, pruned store
//   (k_xbasis2, k_col2p, k_col2: the SPECTRAL_BASIS x pass and the column passes, kernels2.cuh)
//   k_ewald_chi, k_ewald_basis, k_ewald_basis_2d
//                 Ewald gather (Eq. 8) + (I - r r^T) + |.|^2 (Eq. 7) -> (I_xx, I_yy, I_xy, valid)
//   k_rotate_avg  rotate back by -zeta (bilinear), accumulate over angles, divide by counts
// Geometry decisions use IEEE double with explicitly rounded operations (__dmul_rn ...), the
// same sequence DESIGN.md 3-A11 writes out, so validity/cell decisions do not depend on FMA
// contraction.  Values are float32.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "fft_core.cuh"

namespace cyr {

constexpr int MAX_MAT = 32;

// First statement of every kernel of the path.  The host launches them with programmatic dependent launch allowed
// (launch_pdl in cyrsoxs_api.cu): the grid may start while the previous kernel of the stream is still draining.
// griddepcontrol.wait blocks until that kernel has completed and its writes are visible (a no-op for a plain launch);
// launch_dependents lets the NEXT kernel of the stream be scheduled as soon as all CTAs of this one have started.
__device__ __forceinline__ void pdl_entry()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// Bins k in [lo, lo + W) (mod N) of a transformed axis are kept, bin k at slot (k - lo) mod N.
struct Window {
    int N, lo, W;
};
// (every axis may have any length up to 2048, DESIGN 3-A14; powers of two take the FFT kernels)
__host__ __device__ __forceinline__ int win_slot(const Window &w, int k)
{
    const int d = k - w.lo;
    if ((w.N & (w.N - 1)) == 0) return d & (w.N - 1);
    const int r = d % w.N;
    return r < 0 ? r + w.N : r;
}

struct MorphPtrs {
    const float *phi[MAX_MAT];
    const float *S[MAX_MAT];
    const float *theta[MAX_MAT];
    const float *psi[MAX_MAT];
    int n_mat;
};

// ------------------------------------------------------------------------------------------
// x pass, PER_ENERGY algorithm.  One CTA = ROWS consecutive (y, z) rows x one energy.
// Per voxel, with w = phi S and coefficients pre-divided by 4 pi (coef[e][m] = {Cc, Ca, Cb},
// Cc = c/4pi, Ca = (a - c)/4pi, Cb = b/4pi, a = n_perp^2-1, b = n_par^2-n_perp^2, c = n_iso^2-1):
//   chi_xx = sum_m Cc phi + Ca w + Cb w dx dx      chi_xy = sum_m Cb w dx dy
//   chi_yy = sum_m Cc phi + Ca w + Cb w dy dy      chi_xz = sum_m Cb w dx dz
//                                                   chi_yz = sum_m Cb w dy dz
// which is Eq. 5's p for e = x (chi_xx, chi_xy, chi_xz) and e = y (chi_xy, chi_yy, chi_yz).
// Output field f of energy e: out[((e*5 + f) * rows + row) * pitch + slot].
constexpr int NCHI = 5;

template <int LOGN> struct XCfg {
    static constexpr int N = 1 << LOGN;
    static constexpr int TPR = N / 4 > 0 ? N / 4 : 1;                    // threads per row (4 voxels each)
    static constexpr int ROWS = TPR >= 256 ? 1 : 256 / TPR;              // rows per CTA
    static constexpr int THREADS = TPR * ROWS;
    static constexpr int NLINES = ROWS * NCHI;
    static constexpr int LS = RowLayout<N>::LS;
    static constexpr size_t SMEM = sizeof(float) * 2 * (size_t)NLINES * LS + sizeof(float2) * N
                                   + sizeof(float) * 6 * MAX_MAT;
};

template <int LOGN>
__global__ void __launch_bounds__(XCfg<LOGN>::THREADS)
k_xpass_chi(const __grid_constant__ MorphPtrs mp, const float *__restrict__ coef, int e0,
            float2 *__restrict__ out, int rows_total, Window wx, int pitch,
            const float2 *__restrict__ tw_g)
{
    pdl_entry();
    using Cfg = XCfg<LOGN>;
    constexpr int N = Cfg::N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *re = reinterpret_cast<float *>(smem_raw);
    float *im = re + Cfg::NLINES * Cfg::LS;
    float2 *tw = reinterpret_cast<float2 *>(im + Cfg::NLINES * Cfg::LS);
    float *cf = reinterpret_cast<float *>(tw + N);

    const int tid = threadIdx.x;
    const int e = blockIdx.y;
    const int row0 = blockIdx.x * Cfg::ROWS;
    const int nrows = min(Cfg::ROWS, rows_total - row0);
    const int n_mat = mp.n_mat;

    for (int i = tid; i < N; i += Cfg::THREADS) tw[i] = tw_g[i];
    for (int i = tid; i < 6 * n_mat; i += Cfg::THREADS) cf[i] = coef[(size_t)(e0 + e) * 6 * n_mat + i];
    __syncthreads();

    const int rr = tid / Cfg::TPR, tx = tid % Cfg::TPR;
    if (rr < nrows) {
        float acc[4][2 * NCHI];
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
            for (int q = 0; q < 2 * NCHI; ++q) acc[v][q] = 0.f;
        const size_t base = (size_t)(row0 + rr) * N + 4 * tx;
        constexpr int NV = N >= 4 ? 4 : N;
        for (int m = 0; m < n_mat; ++m) {
            const float ccr = cf[6 * m], cci = cf[6 * m + 1], car = cf[6 * m + 2], cai = cf[6 * m + 3],
                        cbr = cf[6 * m + 4], cbi = cf[6 * m + 5];
            float ph[4], s[4], th[4], ps[4];
            const bool aligned = mp.S[m] != nullptr;
            if (N >= 4) {
                float4 t = __ldg(reinterpret_cast<const float4 *>(mp.phi[m] + base));
                ph[0] = t.x; ph[1] = t.y; ph[2] = t.z; ph[3] = t.w;
                if (aligned) {
                    t = __ldg(reinterpret_cast<const float4 *>(mp.S[m] + base));
                    s[0] = t.x; s[1] = t.y; s[2] = t.z; s[3] = t.w;
                    t = __ldg(reinterpret_cast<const float4 *>(mp.theta[m] + base));
                    th[0] = t.x; th[1] = t.y; th[2] = t.z; th[3] = t.w;
                    t = __ldg(reinterpret_cast<const float4 *>(mp.psi[m] + base));
                    ps[0] = t.x; ps[1] = t.y; ps[2] = t.z; ps[3] = t.w;
                }
            } else {
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    ph[v] = mp.phi[m][base + v];
                    if (aligned) { s[v] = mp.S[m][base + v]; th[v] = mp.theta[m][base + v]; ps[v] = mp.psi[m][base + v]; }
                }
            }
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const float f = ph[v];
                float dr = ccr * f, di = cci * f;           // diagonal (isotropic-like) part
                if (aligned) {
                    const float w = f * s[v];
                    float st, ct, sp, cp;
                    sincosf(th[v], &st, &ct);
                    sincosf(ps[v], &sp, &cp);
                    const float dx = cp * st, dy = sp * st, dz = ct;
                    dr = fmaf(car, w, dr); di = fmaf(cai, w, di);
                    const float br = cbr * w, bi = cbi * w;
                    const float xx = dx * dx, yy = dy * dy, xy = dx * dy, xz = dx * dz, yz = dy * dz;
                    acc[v][0] = fmaf(br, xx, acc[v][0]); acc[v][1] = fmaf(bi, xx, acc[v][1]);
                    acc[v][2] = fmaf(br, xy, acc[v][2]); acc[v][3] = fmaf(bi, xy, acc[v][3]);
                    acc[v][4] = fmaf(br, xz, acc[v][4]); acc[v][5] = fmaf(bi, xz, acc[v][5]);
                    acc[v][6] = fmaf(br, yy, acc[v][6]); acc[v][7] = fmaf(bi, yy, acc[v][7]);
                    acc[v][8] = fmaf(br, yz, acc[v][8]); acc[v][9] = fmaf(bi, yz, acc[v][9]);
                }
                acc[v][0] += dr; acc[v][1] += di;
                acc[v][6] += dr; acc[v][7] += di;
            }
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const int p = RowLayout<N>::input_pos(4 * tx + v);
#pragma unroll
            for (int f = 0; f < NCHI; ++f) {
                const int o = (rr * NCHI + f) * Cfg::LS + p;
                re[o] = acc[v][2 * f]; im[o] = acc[v][2 * f + 1];
            }
        }
    }
    __syncthreads();

    RowAcc<N> racc{re, im};
    fft_lines<LOGN, Cfg::NLINES, Cfg::THREADS>(racc, nrows * NCHI, tw, tid);

    // pruned store: slot s <- bin (lo + s) mod N; pad columns [W, pitch) are zeroed
    const int nl = nrows * NCHI;
    const size_t fstride = (size_t)rows_total * pitch;
    for (int idx = tid; idx < nl * pitch; idx += Cfg::THREADS) {
        const int line = idx / pitch, sl = idx - line * pitch;
        const int r = line / NCHI, f = line - r * NCHI;
        float2 val = make_float2(0.f, 0.f);
        if (sl < wx.W) {
            const int b = (wx.lo + sl) & (N - 1);
            const int p = line * Cfg::LS + RowLayout<N>::pos(b);
            val = make_float2(re[p], im[p]);
        }
        out[((size_t)e * NCHI + f) * fstride + (size_t)(row0 + r) * pitch + sl] = val;
    }
}

// ------------------------------------------------------------------------------------------
// SPECTRAL_BASIS algorithm (DESIGN 7.0): p is linear in the optical constants, so the
// energy-independent REAL fields
//   aligned material m:  phi, w = phi S, w dx dx, w dy dy, w dx dy, w dx dz, w dy dz   (7)
//   isotropic material:  phi                                                           (1)
// are transformed once per run (k_xbasis2 in kernels2.cuh).  Two real fields share one complex
// transform (field 2j in the real part of pack j, field 2j+1 in the imaginary part); the Ewald
// kernel separates them with F_a(q) = (Z(q) + conj Z(-q))/2, F_b(q) = (Z(q) - conj Z(-q))/(2i).
enum BasisKind : int { BK_NONE = 0, BK_PHI, BK_W, BK_XX, BK_YY, BK_XY, BK_XZ, BK_YZ };

// ------------------------------------------------------------------------------------------
// Strided pass (z or y), kernels in kernels2.cuh: a CTA transforms a tile of TX contiguous columns by
// N rows and stores the rows whose bins lie in the window.  Batches: blockIdx.x = tile +
// n_tiles * lo, blockIdx.y = hi, with separate in/out strides (in float2 units).
struct ColParams {
    const float2 *in;
    float2 *out;
    int n_tiles;
    long long in_row, out_row;        // stride between consecutive transform indices / slots
    long long in_lo, out_lo;          // stride of the inner batch index (blockIdx.x / n_tiles)
    long long in_hi, out_hi;          // stride of the outer batch index (blockIdx.y)
    Window win;
    const float2 *tw;
};

// ------------------------------------------------------------------------------------------
// Ewald projection.  One thread per detector pixel and energy.
// Image layout shared by the Ewald and rotate kernels ("energy interleaved"): the batch's
// energies are grouped EG at a time (EG = 1, 2, 4 or 8) and the float4 of energy e at pixel
// (iy, ix) sits at  img[(((e / EG) * Ny + iy) * Nx + ix) * EG + e % EG].
// Lanes of a warp run over the EG energies of a group first and over 32 / EG adjacent pixels
// second: the bilinear taps of the rotate kernel, whose position depends on the pixel and the
// angle but not on the energy, then fetch EG * 16 contiguous bytes per pixel (one full 128-byte
// line for EG = 8) instead of 16 bytes from 32 scattered places -- ncu showed that kernel bound
// by L1 wavefronts (14 per 128-bit load, profiles/r1b) -- and the Ewald kernels read the
// spectrum once per pixel for EG energies (same address across the EG lanes: a broadcast).
struct EwaldParams {
    int Nx, Ny, Nz, mode;
    double dqx, dqy, dqz;
    const double *k;            // [n_energy] wavenumbers, nm^-1
    int e0, n_e;                // first energy of the batch, energies in the batch
    Window wx, wy, wz;
    int pitch;                  // x pitch of the spectrum cube
    const float2 *spec;         // [e][f][slot_z][slot_y][pitch]
    float4 *img;                // energy-interleaved (I_xx, I_yy, I_xy, valid)
};

struct PixelGeom {
    int n_nodes;
    int node[2];
    float wt[2];
    float r[3];
};

// DESIGN 3-A5/A8/A11/A13; every double operation is individually rounded.
__device__ __forceinline__ PixelGeom pixel_geometry(int ix, int iy, int Nx, int Ny, int Nz, int mode,
                                                    double dqx, double dqy, double dqz, double k)
{
    PixelGeom g;
    g.n_nodes = 0;
    const double qx = __dmul_rn((double)(ix - Nx / 2), dqx);
    const double qy = __dmul_rn((double)(iy - Ny / 2), dqy);
    const double s2 = __dsub_rn(__dsub_rn(__dmul_rn(k, k), __dmul_rn(qx, qx)), __dmul_rn(qy, qy));
    if (s2 < 0.0) return g;
    const double root = __dsqrt_rn(s2);
    const double qz = __dsub_rn(root, k);
    // r = (q_x, q_y, q_z + k)/k feeds fp32 values only (no decision), so one reciprocal and three
    // multiplications replace three of the kernel's four double divisions; q_z + k is the root itself
    const double ik = __drcp_rn(k);
    g.r[0] = (float)__dmul_rn(qx, ik);
    g.r[1] = (float)__dmul_rn(qy, ik);
    g.r[2] = (float)__dmul_rn(root, ik);
    if (Nz == 1) { g.n_nodes = 1; g.node[0] = 0; g.wt[0] = 1.f; return g; }
    const double gz = __ddiv_rn(qz, dqz);
    if (mode == 0) {
        const double n = floor(__dadd_rn(gz, 0.5));
        if (n < (double)(-(Nz / 2))) return g;
        g.n_nodes = 1; g.node[0] = (int)n; g.wt[0] = 1.f;
        return g;
    }
    const double lo = floor(gz);
    if (lo < (double)(-(Nz / 2))) return g;
    const double t = __dsub_rn(gz, lo);
    int c = 0;
    if (__dsub_rn(1.0, t) > 0.0) { g.node[c] = (int)lo; g.wt[c] = (float)__dsub_rn(1.0, t); ++c; }
    if (t > 0.0) { g.node[c] = (int)lo + 1; g.wt[c] = (float)t; ++c; }
    g.n_nodes = c;
    return g;
}

// (I - r r^T) applied to p~ for e = x (u) and e = y (v); returns |.|^2, |.|^2, Re<.,.>.
__device__ __forceinline__ void project_pair(const float r[3], const float2 u[3], const float2 v[3],
                                             float &sxx, float &syy, float &sxy)
{
    float2 ru = make_float2(r[0] * u[0].x + r[1] * u[1].x + r[2] * u[2].x, r[0] * u[0].y + r[1] * u[1].y + r[2] * u[2].y);
    float2 rv = make_float2(r[0] * v[0].x + r[1] * v[1].x + r[2] * v[2].x, r[0] * v[0].y + r[1] * v[1].y + r[2] * v[2].y);
    sxx = syy = sxy = 0.f;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const float2 wu = make_float2(u[d].x - r[d] * ru.x, u[d].y - r[d] * ru.y);
        const float2 wv = make_float2(v[d].x - r[d] * rv.x, v[d].y - r[d] * rv.y);
        sxx += wu.x * wu.x + wu.y * wu.y;
        syy += wv.x * wv.x + wv.y * wv.y;
        sxy += wu.x * wv.x + wu.y * wv.y;
    }
}

// Thread mapping of both Ewald kernels: 256 threads = 256 / EG pixels x EG energies.
template <int EG> struct EwaldMap {
    static constexpr int P = 256 / EG;                 // pixels per CTA
    static constexpr int PW = P >= 32 ? 32 : P;        // ... as PW x PH
    static constexpr int PH = P / PW;
};

template <int EG>
__global__ void __launch_bounds__(256)
k_ewald_chi(const EwaldParams p)
{
    pdl_entry();
    using M = EwaldMap<EG>;
    const int sub = threadIdx.x % EG, pp = threadIdx.x / EG;
    const int ix = blockIdx.x * M::PW + pp % M::PW;
    const int iy = blockIdx.y * M::PH + pp / M::PW;
    const int e = blockIdx.z * EG + sub;
    if (ix >= p.Nx || iy >= p.Ny) return;
    float axx = 0.f, ayy = 0.f, axy = 0.f;
    bool valid = false;
    if (e < p.n_e) {
        const double k = p.k[p.e0 + e];
        const PixelGeom g = pixel_geometry(ix, iy, p.Nx, p.Ny, p.Nz, p.mode, p.dqx, p.dqy, p.dqz, k);
        valid = g.n_nodes > 0;
        if (valid) {
            const int sx = win_slot(p.wx, ix - p.Nx / 2), sy = win_slot(p.wy, iy - p.Ny / 2);
            const size_t plane = (size_t)p.wy.W * p.pitch;
            const size_t fstride = plane * p.wz.W;
            const float2 *base = p.spec + (size_t)e * NCHI * fstride + (size_t)sy * p.pitch + sx;
            const double k2 = k * k;
            const float k4 = (float)(k2 * k2);
            const bool inwin = sx < p.wx.W && sy < p.wy.W;
            for (int j = 0; j < g.n_nodes; ++j) {
                const int sz = win_slot(p.wz, g.node[j]);
                float2 c[NCHI];
#pragma unroll
                for (int f = 0; f < NCHI; ++f)
                    c[f] = (inwin && sz < p.wz.W) ? __ldg(base + f * fstride + (size_t)sz * plane) : make_float2(0.f, 0.f);
                const float2 u[3] = {c[0], c[1], c[2]}, v[3] = {c[1], c[3], c[4]};
                float sxx, syy, sxy;
                project_pair(g.r, u, v, sxx, syy, sxy);
                const float w = g.wt[j] * k4;
                axx = fmaf(w, sxx, axx); ayy = fmaf(w, syy, ayy); axy = fmaf(w, sxy, axy);
            }
        }
    }
    p.img[(((size_t)blockIdx.z * p.Ny + iy) * p.Nx + ix) * EG + sub] = make_float4(axx, ayy, axy, valid ? 1.f : 0.f);
}

// Ewald projection for SPECTRAL_BASIS: chi~(q) = sum_b coef[e][b] F_b(q) on the shell only.
struct EwaldBasisParams {
    EwaldParams g;              // geometry, windows, spec = packed spectra [pack][wz][wy][pitch], img
    int n_pack;
    const float2 *coef;         // [n_energy][2 n_pack], already multiplied by 1/2 (the unpacking factor)
    const int *kind;            // [2 n_pack] BasisKind
};

#ifndef CYRSOXS_EW_PU
#define CYRSOXS_EW_PU 4
#endif
constexpr int EW_PU = CYRSOXS_EW_PU;        // packs gathered per chunk in k_ewald_basis

template <int EG>
__global__ void __launch_bounds__(256)
k_ewald_basis(const EwaldBasisParams q)
{
    pdl_entry();
    using M = EwaldMap<EG>;
    const EwaldParams &p = q.g;
    const int sub = threadIdx.x % EG, pp = threadIdx.x / EG;
    const int ix = blockIdx.x * M::PW + pp % M::PW;
    const int iy = blockIdx.y * M::PH + pp / M::PW;
    const int e = blockIdx.z * EG + sub;
    if (ix >= p.Nx || iy >= p.Ny) return;
    float axx = 0.f, ayy = 0.f, axy = 0.f;
    bool valid = false;
    if (e < p.n_e) {
        const double k = p.k[p.e0 + e];
        const PixelGeom g = pixel_geometry(ix, iy, p.Nx, p.Ny, p.Nz, p.mode, p.dqx, p.dqy, p.dqz, k);
        valid = g.n_nodes > 0;
        if (valid) {
            const int mx = ix - p.Nx / 2, my = iy - p.Ny / 2;
            const int sx = win_slot(p.wx, mx), sy = win_slot(p.wy, my);
            const int tx = win_slot(p.wx, -mx), ty = win_slot(p.wy, -my);
            const size_t plane = (size_t)p.wy.W * p.pitch;
            const size_t fstride = plane * p.wz.W;
            const bool inwin = sx < p.wx.W && sy < p.wy.W && tx < p.wx.W && ty < p.wy.W;
            const double k2 = k * k;
            const float k4 = (float)(k2 * k2);
            const float2 *coef = q.coef + (size_t)(p.e0 + e) * 2 * q.n_pack;
            for (int j = 0; j < g.n_nodes; ++j) {
                const int sz = win_slot(p.wz, g.node[j]), tz = win_slot(p.wz, -g.node[j]);
                const bool ok = inwin && sz < p.wz.W && tz < p.wz.W;
                const float2 *pq = p.spec + (size_t)sz * plane + (size_t)sy * p.pitch + sx;      // advanced pack by pack
                const float2 *pm = p.spec + (size_t)tz * plane + (size_t)ty * p.pitch + tx;
                float2 c[NCHI];
#pragma unroll
                for (int f = 0; f < NCHI; ++f) c[f] = make_float2(0.f, 0.f);
                // EW_PU packs at a time: the gathers of a chunk are issued before the first is used (the kernel is bound by the
                // latency of these L2 gathers, ncu: long scoreboard 9 cycles per issue); same summation order.  Measured
                // (CFG3 / CFG5 Ewald stage): one pack at a time 0.365 / 0.49 ms, four 0.314 / 0.406 ms; both nodes at once on
                // top of that (120 registers, 2 CTAs per SM) 0.367 / 0.529 ms.
                for (int pk0 = 0; ok && pk0 < q.n_pack; pk0 += EW_PU, pq += EW_PU * fstride, pm += EW_PU * fstride) {
                    float2 z1[EW_PU], z2[EW_PU];
#pragma unroll
                    for (int u = 0; u < EW_PU; ++u) {
                        const bool have = pk0 + u < q.n_pack;
                        z1[u] = have ? __ldg(pq + u * fstride) : make_float2(0.f, 0.f);
                        z2[u] = have ? __ldg(pm + u * fstride) : make_float2(0.f, 0.f);
                    }
#pragma unroll
                    for (int u = 0; u < EW_PU; ++u) {
                        const int pk = pk0 + u;
                        // Fa = z1 + conj z2, Fb = -i (z1 - conj z2)   (the 1/2 lives in coef)
                        const float2 F[2] = {make_float2(z1[u].x + z2[u].x, z1[u].y - z2[u].y), make_float2(z1[u].y + z2[u].y, z2[u].x - z1[u].x)};
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            if (pk >= q.n_pack) continue;                      // (uniform: the padding of the last chunk)
                            const int kd = __ldg(q.kind + 2 * pk + h);
                            const float2 v = cmul(__ldg(coef + 2 * pk + h), F[h]);
                            if (kd == BK_PHI || kd == BK_W) { c[0] = cadd(c[0], v); c[3] = cadd(c[3], v); }
                            else if (kd == BK_XX) c[0] = cadd(c[0], v);
                            else if (kd == BK_YY) c[3] = cadd(c[3], v);
                            else if (kd == BK_XY) c[1] = cadd(c[1], v);
                            else if (kd == BK_XZ) c[2] = cadd(c[2], v);
                            else if (kd == BK_YZ) c[4] = cadd(c[4], v);
                        }
                    }
                }
                const float2 u[3] = {c[0], c[1], c[2]}, v[3] = {c[1], c[3], c[4]};
                float sxx, syy, sxy;
                project_pair(g.r, u, v, sxx, syy, sxy);
                const float w = g.wt[j] * k4;
                axx = fmaf(w, sxx, axx); ayy = fmaf(w, syy, ayy); axy = fmaf(w, sxy, axy);
            }
        }
    }
    p.img[(((size_t)blockIdx.z * p.Ny + iy) * p.Nx + ix) * EG + sub] = make_float4(axx, ayy, axy, valid ? 1.f : 0.f);
}

// Ewald projection for SPECTRAL_BASIS on a 2-D model (Nz = 1, A13): the k_z = 0 plane serves every energy, so a thread
// owns one pixel, gathers and unpacks its basis spectra once and loops over the batch's energies; per energy only the
// validity and r-hat (fp64, same operation order as pixel_geometry), the coefficient sum and the projection remain.
// The unpacked fields F_b of the pixel sit in shared memory ([field][thread], conflict-free 64-bit accesses), which lets
// the coefficient sum walk the basis MATERIAL BY MATERIAL (an aligned material is the run PHI, W, XX, YY, XY, XZ, YZ, an
// isotropic one a single PHI; the kind table is only read to tell the two apart) with no per-field dispatch: round 1's
// version kept F in registers, which forces compile-time field indices and a kind test per field and energy -- 388
// thread-instructions per pixel and energy, 75 % of the issue slots (ncu r2_cfg4).  Coefficients, k, 1/k and k^4 of the
// batch sit in shared memory too.  Same additions in the same order as k_ewald_basis: identical images.
constexpr int EW2D_MAXF = 64;          // most basis fields (2 n_pack) the shared-memory layout is sized for

template <int EG>
__global__ void __launch_bounds__(256)
k_ewald_basis_2d(const EwaldBasisParams q)
{
    pdl_entry();
    const EwaldParams &p = q.g;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nb = 2 * q.n_pack, ne = p.n_e;
    double *s_k = reinterpret_cast<double *>(smem_raw);              // [ne] k, then [ne] 1/k
    double *s_ik = s_k + ne;
    float2 *s_coef = reinterpret_cast<float2 *>(s_ik + ne);          // [ne][nb]
    float2 *s_F = s_coef + (size_t)ne * nb;                           // [nb][256]
    float *s_k4 = reinterpret_cast<float *>(s_F + (size_t)nb * 256);  // [ne]
    int *s_kind = reinterpret_cast<int *>(s_k4 + ne);                 // [nb]
    for (int e = threadIdx.x; e < ne; e += 256) {
        const double k = p.k[p.e0 + e];
        s_k[e] = k; s_ik[e] = __drcp_rn(k);
        const double k2 = k * k;
        s_k4[e] = (float)(k2 * k2);
    }
    for (int i = threadIdx.x; i < ne * nb; i += 256) s_coef[i] = q.coef[(size_t)p.e0 * nb + i];
    for (int i = threadIdx.x; i < nb; i += 256) s_kind[i] = q.kind[i];
    const int tid = threadIdx.x;
    const int ix = blockIdx.x * 32 + (tid & 31);
    const int iy = blockIdx.y * 8 + (tid >> 5);
    const bool inside = ix < p.Nx && iy < p.Ny;
    const int mx = ix - p.Nx / 2, my = iy - p.Ny / 2;
    const int sx = win_slot(p.wx, mx), sy = win_slot(p.wy, my);
    const int tx = win_slot(p.wx, -mx), ty = win_slot(p.wy, -my);
    const bool inwin = inside && sx < p.wx.W && sy < p.wy.W && tx < p.wx.W && ty < p.wy.W;
    const size_t fstride = (size_t)p.wy.W * p.pitch;                 // wz.W == 1
    const float2 *pq = p.spec + (size_t)sy * p.pitch + sx;
    const float2 *pm = p.spec + (size_t)ty * p.pitch + tx;
    float2 *F = s_F + tid;                                            // field b of this pixel at F[b * 256]
    for (int pk0 = 0; pk0 < q.n_pack; pk0 += EW_PU) {                 // EW_PU packs' gathers in flight
        float2 z1[EW_PU], z2[EW_PU];
#pragma unroll
        for (int u = 0; u < EW_PU; ++u) {
            const bool have = inwin && pk0 + u < q.n_pack;
            z1[u] = have ? __ldg(pq + (size_t)(pk0 + u) * fstride) : make_float2(0.f, 0.f);
            z2[u] = have ? __ldg(pm + (size_t)(pk0 + u) * fstride) : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < EW_PU; ++u) {
            if (pk0 + u < q.n_pack) {
                // Fa = z1 + conj z2, Fb = -i (z1 - conj z2)   (the 1/2 lives in coef)
                F[(2 * (pk0 + u)) * 256] = make_float2(z1[u].x + z2[u].x, z1[u].y - z2[u].y);
                F[(2 * (pk0 + u) + 1) * 256] = make_float2(z1[u].y + z2[u].y, z2[u].x - z1[u].x);
            }
        }
    }
    __syncthreads();                                                  // the tables (F itself is private to the thread)
    if (!inside) return;
    const double qx = __dmul_rn((double)mx, p.dqx), qy = __dmul_rn((double)my, p.dqy);
    const double qx2 = __dmul_rn(qx, qx), qy2 = __dmul_rn(qy, qy);
    const size_t pix = (size_t)iy * p.Nx + ix, plane = (size_t)p.Ny * p.Nx;
    for (int e = 0; e < ne; ++e) {
        const double k = s_k[e];
        const double s2 = __dsub_rn(__dsub_rn(__dmul_rn(k, k), qx2), qy2);
        float4 res = make_float4(0.f, 0.f, 0.f, 0.f);
        if (s2 >= 0.0) {
            const double ik = s_ik[e];
            const float r[3] = {(float)__dmul_rn(qx, ik), (float)__dmul_rn(qy, ik), (float)__dmul_rn(__dsqrt_rn(s2), ik)};
            float2 c0 = make_float2(0.f, 0.f), c1 = c0, c2 = c0, c3 = c0, c4 = c0;
            const float2 *coef = s_coef + (size_t)e * nb;
            if (inwin) {
                for (int b = 0; b < nb;) {
                    const int kd = s_kind[b];
                    if (kd == BK_NONE) { ++b; continue; }                         // padding of a pack / of a material group
                    const bool aligned = b + 1 < nb && s_kind[b + 1] == BK_W;      // kd == BK_PHI starts a material
                    float2 v = cmul(coef[b], F[b * 256]);                         // PHI
                    c0 = cadd(c0, v); c3 = cadd(c3, v);
                    if (aligned) {
                        v = cmul(coef[b + 1], F[(b + 1) * 256]); c0 = cadd(c0, v); c3 = cadd(c3, v);      // W
                        c0 = cadd(c0, cmul(coef[b + 2], F[(b + 2) * 256]));                                // XX
                        c3 = cadd(c3, cmul(coef[b + 3], F[(b + 3) * 256]));                                // YY
                        c1 = cadd(c1, cmul(coef[b + 4], F[(b + 4) * 256]));                                // XY
                        c2 = cadd(c2, cmul(coef[b + 5], F[(b + 5) * 256]));                                // XZ
                        c4 = cadd(c4, cmul(coef[b + 6], F[(b + 6) * 256]));                                // YZ
                        b += 7;
                    } else ++b;
                }
            }
            const float2 u[3] = {c0, c1, c2}, v3[3] = {c1, c3, c4};
            float sxx, syy, sxy;
            project_pair(r, u, v3, sxx, syy, sxy);
            const float w = 1.f * s_k4[e];
            res = make_float4(fmaf(w, sxx, 0.f), fmaf(w, syy, 0.f), fmaf(w, sxy, 0.f), 1.f);
        }
        p.img[((size_t)(e / EG) * plane + pix) * EG + e % EG] = res;
    }
}

// ------------------------------------------------------------------------------------------
// Rotate back and average (DESIGN 3-A9/A10).  A thread owns one output pixel and one energy of
// every energy group (lanes: EG energies x 32/EG pixels, see EwaldParams).  The bilinear cell
// of an (output pixel, angle) pair is pure geometry (fp64, every operation rounded on its own)
// and does not depend on the energy: it is computed once per angle and reused for all groups.
// cs[a] = (C, S) in double; csf[a] = (C^2, S^2, 2 C S).
//  * tiles are visited in order of their distance from q = 0 (table built on the host): the CTAs
//    resident at one time cover an annulus, and the source pixels of an annulus are the same
//    annulus at every angle, so an image is read from DRAM about once instead of once per angle;
//  * all 4 UA loads of an angle chunk are issued before the first use.
struct RotateParams {
    int Nx, Ny, n_angles, n_energy;
    const double2 *cs;
    const float4 *csf;
    const float4 *img;          // energy-interleaved, see EwaldParams
    float *out;                 // [e][Ny][Nx]
    unsigned int *counts;       // optional
    const float *reach2;        // [e] squared reach (in pixels of x) of the valid disk, see below
    const uint32_t *tiles;      // [n_tiles] (tile_y << 16 | tile_x), sorted by distance from q = 0
    double rho;                 // Nx / Ny
    int gpc;                    // energy groups per CTA (blockIdx.y slices the groups)
};

// 256 threads = AS angle slices x WS = 8 / AS warps; the WS warps of a slice tile WSX x WSY warp
// patches, a warp covers WPW x WPH pixels times EG energies.  AS > 1 (small images: too few
// tiles to fill the machine, and every thread a long serial chain over the angles) gives every
// pixel AS threads that each take a contiguous share of the angles; their partial sums are added
// in slice order at the end, so the result does not depend on scheduling.
template <int EG, int AS> struct RotMap {
    static constexpr int WP = 32 / EG;                                        // pixels per warp
    static constexpr int WPW = WP >= 16 ? 8 : (WP == 8 ? 4 : 2);              // 8x4, 8x2, 4x2, 2x2
    static constexpr int WPH = WP / WPW;
    static constexpr int WS = 8 / AS;                                         // warps per slice
    static constexpr int WSX = WS >= 4 ? (WS == 8 ? 4 : 2) : WS;              // 4x2, 2x2, 2x1, 1x1
    static constexpr int WSY = WS / WSX;
    static constexpr int TW = WSX * WPW, TH = WSY * WPH;                      // CTA tile
};

// reach2[e] = (k_e/dq_x + sqrt(1 + rho^2) + 1)^2 (+ 0.01 %): an output pixel whose distance from q = 0 (measured in x
// pixels, y pixels scaled by rho) exceeds the reach has every bilinear neighbour outside the
// Ewald disk s^2 >= 0 at every angle (rotation keeps the distance, a cell adds < 2 pixels), so
// its count is 0 and nothing needs to be read.  The margin (cell diagonal + 1) keeps the decision away from
// rounding: only pixels that are invalid with certainty are skipped.
//
// Loop order: angles in chunks of UA; the chunk's cells are computed once (registers) and
// then applied to every energy group of the CTA's slice (blockIdx.y, gpc <= ROT_GMAX groups),
// whose running sums and counts live in shared memory between chunks.
constexpr int ROT_GMAX = 16;      // most energy groups per CTA (RotateParams::gpc <= ROT_GMAX)

template <int EG, int UA, int MINB, int AS>
__global__ void __launch_bounds__(256, MINB)
k_rotate_avg(const RotateParams p)
{
    pdl_entry();
    using M = RotMap<EG, AS>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n_groups = (p.n_energy + EG - 1) / EG;
    const int g0 = blockIdx.y * p.gpc;
    const int ng = min(min(p.gpc, ROT_GMAX), n_groups - g0);
    float *s_sum = reinterpret_cast<float *>(smem_raw);                       // [ng][256]
    unsigned int *s_cnt = reinterpret_cast<unsigned int *>(s_sum + ng * 256);  // [ng][256]
    const uint32_t tile = __ldg(p.tiles + blockIdx.x);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sub = lane % EG, lp = lane / EG;
    const int slice = warp / M::WS, wl = warp % M::WS;
    const int ix = (int)(tile & 0xffffu) * M::TW + (wl % M::WSX) * M::WPW + lp % M::WPW;
    const int iy = (int)(tile >> 16) * M::TH + (wl / M::WSX) * M::WPH + lp / M::WPW;
    const bool inside = ix < p.Nx && iy < p.Ny;
    if (AS == 1 && !inside) return;                             // AS == 1: no block-wide barrier below
    const size_t plane = (size_t)p.Ny * p.Nx * EG;               // float4 per energy group
    const float4 *img = p.img + (size_t)g0 * plane + sub;
    const double rho = p.rho;
    const double u = (double)(ix - p.Nx / 2), v = (double)(iy - p.Ny / 2);
    const double vr = v * rho, ur = u / rho;                 // each rounded once, as in the oracle (rho = Nx/Ny need not be a power of two)
    const double cx = (double)(p.Nx / 2), cy = (double)(p.Ny / 2);
    const double xmax = (double)(p.Nx - 1), ymax = (double)(p.Ny - 1);
    const float r2 = (float)(u * u + vr * vr);
    // live groups of this lane: bit j <=> energy (g0 + j) EG + sub exists and the pixel is within its reach
    unsigned int live = 0;
    for (int j = 0; j < ng; ++j) {
        const int e = (g0 + j) * EG + sub;
        if (inside && e < p.n_energy && r2 <= __ldg(p.reach2 + e)) live |= 1u << j;
        s_sum[j * 256 + tid] = 0.f;
        s_cnt[j * 256 + tid] = 0u;
    }
    // this slice's share of the angles: [a_begin, na)
    const int per = (p.n_angles + AS - 1) / AS;
    const int a_begin = slice * per;
    const int na = live ? min(p.n_angles, a_begin + per) : 0;
    const int rowq = p.Nx * EG;
    for (int a0 = a_begin; a0 < na; a0 += UA) {
        int o00[UA], o10[UA], o01[UA], o11[UA];          // element offsets of the four taps within a group
        float w00[UA], w10[UA], w01[UA], w11[UA], wx[UA], wy[UA], wz[UA];
        bool ok[UA];
#pragma unroll
        for (int q = 0; q < UA; ++q) {
            const int a = min(a0 + q, na - 1);
            const double2 cs = __ldg(p.cs + a);
            const float4 w = __ldg(p.csf + a);
            wx[q] = w.x; wy[q] = w.y; wz[q] = w.z;
            const double fx = __dadd_rn(__dsub_rn(__dmul_rn(cs.x, u), __dmul_rn(cs.y, vr)), cx);
            const double fy = __dadd_rn(__dadd_rn(__dmul_rn(cs.y, ur), __dmul_rn(cs.x, v)), cy);
            const double x0 = floor(fx), y0 = floor(fy);
            const double al = fx - x0, be = fy - y0;
            const int dx = al > 0.0 ? 1 : 0, dy = be > 0.0 ? 1 : 0;    // a neighbour is needed iff its weight > 0
            ok[q] = (a0 + q < na) && !(x0 < 0.0 || y0 < 0.0 || x0 + (double)dx > xmax || y0 + (double)dy > ymax);
            // un-needed neighbours alias a needed one (weight 0, same validity)
            o00[q] = ok[q] ? ((int)y0 * p.Nx + (int)x0) * EG : 0;
            const int ox = ok[q] ? dx * EG : 0, oy = ok[q] ? dy * rowq : 0;
            o10[q] = o00[q] + ox; o01[q] = o00[q] + oy; o11[q] = o01[q] + ox;
            const float fa = (float)al, fb = (float)be;
            w00[q] = (1.f - fa) * (1.f - fb); w10[q] = fa * (1.f - fb); w01[q] = (1.f - fa) * fb; w11[q] = fa * fb;
        }
        // the groups of this CTA: base pointer, running sums and live bits advance by increments
        // (no per-group multiplications: address arithmetic was a third of the kernel's instructions)
        const float4 *base = img;
        float *ps = s_sum + tid;
        unsigned int *pc = s_cnt + tid;
        unsigned int lv = live;
        for (int j = 0; j < ng; ++j, base += plane, ps += 256, pc += 256, lv >>= 1) {
            if (!(lv & 1u)) continue;
            float4 t[UA][4];
#pragma unroll
            for (int q = 0; q < UA; ++q) {
                t[q][0] = __ldg(base + o00[q]); t[q][1] = __ldg(base + o10[q]);
                t[q][2] = __ldg(base + o01[q]); t[q][3] = __ldg(base + o11[q]);
            }
            float sum = *ps;
            unsigned int cnt = *pc;
#pragma unroll
            for (int q = 0; q < UA; ++q) {
                const float4 t00 = t[q][0], t10 = t[q][1], t01 = t[q][2], t11 = t[q][3];
                const bool good = ok[q] & (t00.w != 0.f) & (t10.w != 0.f) & (t01.w != 0.f) & (t11.w != 0.f);
                float acc = w00[q] * (wx[q] * t00.x + wy[q] * t00.y + wz[q] * t00.z);
                acc = fmaf(w10[q], wx[q] * t10.x + wy[q] * t10.y + wz[q] * t10.z, acc);
                acc = fmaf(w01[q], wx[q] * t01.x + wy[q] * t01.y + wz[q] * t01.z, acc);
                acc = fmaf(w11[q], wx[q] * t11.x + wy[q] * t11.y + wz[q] * t11.z, acc);
                if (good) { sum += acc; ++cnt; }
            }
            *ps = sum;
            *pc = cnt;
        }
    }
    if (AS > 1) __syncthreads();
    if (slice != 0 || !inside) return;
    for (int j = 0; j < ng; ++j) {
        const int e = (g0 + j) * EG + sub;
        if (e < p.n_energy) {
            const size_t o = ((size_t)e * p.Ny + iy) * p.Nx + ix;
            float sum = s_sum[j * 256 + tid];
            unsigned int cnt = s_cnt[j * 256 + tid];
#pragma unroll
            for (int sl = 1; sl < AS; ++sl) {
                sum += s_sum[j * 256 + tid + sl * M::WS * 32];
                cnt += s_cnt[j * 256 + tid + sl * M::WS * 32];
            }
            p.out[o] = cnt ? sum / (float)cnt : 0.f;
            if (p.counts) p.counts[o] = cnt;
        }
    }
}

} // namespace cyr
