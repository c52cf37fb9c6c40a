// reduce.cuh -- 1-D reductions of finished detector images (cyrsoxs_reduce):
// azimuthal average I(|q|), sector anisotropy A, integrated scattering intensity ISI.
//   k_reduce_accumulate  one CTA per (row slab, energy): per-bin sums in shared memory
//                        (double atomics), then one global double atomic per touched bin
//   k_reduce_finalize    means, anisotropy, ISI scale
// Bin and sector decisions are fp64 with individually rounded operations (same order as the
// definition in include/cyrsoxs.h), so a pixel never lands in a different bin than the oracle's.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cyr {

struct ReduceParams {
    int Nx, Ny, n_bins, rows_per_cta;
    double rho, tan_w;
    const float *img;              // [e][Ny][Nx]
    const unsigned int *cnt;       // [e][Ny][Nx] or nullptr
    double *acc;                   // [e][3][n_bins] sums (all, para, perp) then [e] total at the end
    unsigned int *num;             // [e][3][n_bins] pixel counts
    double *total;                 // [e]
};

__global__ void __launch_bounds__(256)
k_reduce_accumulate(const ReduceParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *s_sum = reinterpret_cast<double *>(smem_raw);                         // [3][n_bins]
    unsigned int *s_num = reinterpret_cast<unsigned int *>(s_sum + 3 * p.n_bins);  // [3][n_bins]
    __shared__ double s_total;
    const int e = blockIdx.y, B = p.n_bins;
    for (int i = threadIdx.x; i < 3 * B; i += blockDim.x) { s_sum[i] = 0.0; s_num[i] = 0u; }
    if (threadIdx.x == 0) s_total = 0.0;
    __syncthreads();
    const size_t plane = (size_t)p.Nx * p.Ny;
    const float *img = p.img + (size_t)e * plane;
    const unsigned int *cnt = p.cnt ? p.cnt + (size_t)e * plane : nullptr;
    const int y0 = blockIdx.x * p.rows_per_cta, y1 = min(p.Ny, y0 + p.rows_per_cta);
    double mine = 0.0;
    for (int iy = y0; iy < y1; ++iy) {
        const double v = __dmul_rn((double)(iy - p.Ny / 2), p.rho);
        for (int ix = threadIdx.x; ix < p.Nx; ix += blockDim.x) {
            const size_t o = (size_t)iy * p.Nx + ix;
            if (cnt && __ldg(cnt + o) == 0u) continue;
            const double val = (double)__ldg(img + o);
            mine += val;
            const double u = (double)(ix - p.Nx / 2);
            const double r = __dsqrt_rn(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v)));
            const double fb = floor(__dadd_rn(r, 0.5));
            if (fb >= (double)B) continue;
            const int b = (int)fb;
            atomicAdd(&s_sum[b], val); atomicAdd(&s_num[b], 1u);
            if (u == 0.0 && v == 0.0) continue;
            if (fabs(v) <= __dmul_rn(p.tan_w, fabs(u))) { atomicAdd(&s_sum[B + b], val); atomicAdd(&s_num[B + b], 1u); }
            if (fabs(u) <= __dmul_rn(p.tan_w, fabs(v))) { atomicAdd(&s_sum[2 * B + b], val); atomicAdd(&s_num[2 * B + b], 1u); }
        }
    }
    // warp-reduce the ISI partial, one shared atomic per warp
    for (int d = 16; d > 0; d >>= 1) mine += __shfl_down_sync(0xffffffffu, mine, d);
    if ((threadIdx.x & 31) == 0) atomicAdd(&s_total, mine);
    __syncthreads();
    double *acc = p.acc + (size_t)e * 3 * B;
    unsigned int *num = p.num + (size_t)e * 3 * B;
    for (int i = threadIdx.x; i < 3 * B; i += blockDim.x)
        if (s_num[i]) { atomicAdd(acc + i, s_sum[i]); atomicAdd(num + i, s_num[i]); }
    if (threadIdx.x == 0) atomicAdd(p.total + e, s_total);
}

__global__ void k_reduce_finalize(int n_energy, int n_bins, const double *acc, const unsigned int *num, const double *total,
                                  double dq2, float *I, float *A, float *isi)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_energy * n_bins) return;
    const int e = i / n_bins, b = i - e * n_bins;
    const double *a = acc + (size_t)e * 3 * n_bins;
    const unsigned int *n = num + (size_t)e * 3 * n_bins;
    I[i] = n[b] ? (float)(a[b] / (double)n[b]) : 0.f;
    if (A) {
        float val = 0.f;
        if (n[n_bins + b] && n[2 * n_bins + b]) {
            const double ip = a[n_bins + b] / (double)n[n_bins + b], iq = a[2 * n_bins + b] / (double)n[2 * n_bins + b];
            if (ip + iq != 0.0) val = (float)((ip - iq) / (ip + iq));
        }
        A[i] = val;
    }
    if (isi && b == 0) isi[e] = (float)(total[e] * dq2);
}

// De-interleaves the paper's Real4 morphology of one material into four arrays and
// records max |S| (as the bit pattern of a non-negative float, so an integer atomicMax orders it).
__global__ void __launch_bounds__(256)
k_aos_to_soa(const float4 *__restrict__ src, float *__restrict__ phi, float *__restrict__ S, float *__restrict__ theta,
             float *__restrict__ psi, size_t n, unsigned int *max_s_bits)
{
    float m = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float4 v = __ldcs(src + i);
        phi[i] = v.x; S[i] = v.y; psi[i] = v.z; theta[i] = v.w;
        m = fmaxf(m, fabsf(v.y));
        if (v.y != v.y) m = __int_as_float(0x7f800000);          // NaN counts as "aligned"
    }
    for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_down_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(max_s_bits, __float_as_uint(m));
}

} // namespace cyr
