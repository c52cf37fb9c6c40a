// kernels2.cuh -- second-generation FFT passes built on fft_reg.cuh / fft2.cuh (register-first /
// register-last): the strided z / y passes (k_col2, k_col2p), the SPECTRAL_BASIS x passes (k_xbasis3; k_xbasis2
// below 64 points) and the direct-DFT passes for lengths that are not powers of two (k_coldft, k_xdft).
#pragma once
#include "fft_reg.cuh"
#include "fft2.cuh"
#include "kernels.cuh"

namespace cyr {

// ------------------------------------------------------------------------------------------
// Strided pass (z or y).  A CTA transforms a tile of TX adjacent columns (contiguous along x)
// by N rows of one (lo, hi) batch item.  Thread (li, c): c = tid % TX is the column, li the
// butterfly index.  Loads go straight from global memory into the stage-0 registers (lanes
// run along x: TX * 8 contiguous bytes per row), the last stage stores straight to global,
// pruned to the window.  Same parameters and batch mapping as k_colpass (ColParams).
template <int LOGN> struct Col2Cfg {
    static constexpr int N = 1 << LOGN;
    static constexpr int TX = N <= 256 ? 16 : (N <= 1024 ? 8 : 4);
    using F = RegFft<LOGN, ColMap<TX>>;
    static constexpr int T = F::T;
    static constexpr int THREADS = T * TX;
    static constexpr size_t SMEM = F::NST > 1 ? sizeof(float2) * (size_t)N * TX : 0;
};

template <int LOGN>
__global__ void __launch_bounds__(Col2Cfg<LOGN>::THREADS)
k_col2(const ColParams p)
{
    pdl_entry();
    using Cfg = Col2Cfg<LOGN>;
    using F = typename Cfg::F;
    constexpr int N = Cfg::N, TX = Cfg::TX, T = Cfg::T, R0 = F::R0, NST = F::NST;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *sm = reinterpret_cast<float2 *>(smem_raw);
    const int tid = threadIdx.x;
    const int c = tid % TX, li = tid / TX;
    const int tile = blockIdx.x % p.n_tiles, lo = blockIdx.x / p.n_tiles, hi = blockIdx.y;

    const float2 *src = p.in + (size_t)hi * p.in_hi + (size_t)lo * p.in_lo + (size_t)tile * TX + c;
    float2 v[R0];
#pragma unroll
    for (int s = 0; s < R0; ++s) v[s] = __ldcs(src + (size_t)(li + s * T) * p.in_row);
    F::stage0(v);
    float2 *L = sm + c;
    if constexpr (NST > 1) {
        F::stage0_store(L, li, v);
        float2 w[R0];
        if constexpr (NST > 2) {
            __syncthreads();
            F::template load_tw<1>(p.tw, li, w);
            F::template stage_load<1>(L, li, w, v);
            __syncthreads();
            F::template stage_store<1>(L, li, v);
        }
        if constexpr (NST > 3) {
            __syncthreads();
            F::template load_tw<2>(p.tw, li, w);
            F::template stage_load<2>(L, li, w, v);
            __syncthreads();
            F::template stage_store<2>(L, li, v);
        }
        __syncthreads();
        F::template load_tw<NST - 1>(p.tw, li, w);
        F::template stage_load<NST - 1>(L, li, w, v);
    }
    float2 *dst = p.out + (size_t)hi * p.out_hi + (size_t)lo * p.out_lo + (size_t)tile * TX + c;
#pragma unroll
    for (int m = 0; m < R0; ++m) {
        const int k = li + T * m;
        const int sl = (k - p.win.lo) & (N - 1);
        if (sl < p.win.W) dst[(size_t)sl * p.out_row] = v[F::out_reg(m)];
    }
}

// Same pass with two adjacent columns per thread (128-bit global loads and stores, float4 in shared
// memory): a tile is 16 columns = 128-byte row segments at half the threads of k_col2's 16-column
// configuration.  Used where k_col2 would otherwise fall back to 8-column tiles (N = 512).
template <int LOGN, int PW_> struct Col2PCfg {
    static constexpr int N = 1 << LOGN;
    static constexpr int PW = PW_, TX = 2 * PW;
    using F = RegFft<LOGN, PairMap<PW>>;
    static constexpr int T = F::T;
    static constexpr int THREADS = T * PW;
    static constexpr size_t SMEM = sizeof(float4) * (size_t)N * PW;
};

template <int LOGN, int PW_>
__global__ void __launch_bounds__(Col2PCfg<LOGN, PW_>::THREADS)
k_col2p(const ColParams p)
{
    pdl_entry();
    using Cfg = Col2PCfg<LOGN, PW_>;
    using F = typename Cfg::F;
    constexpr int N = Cfg::N, TX = Cfg::TX, PW = Cfg::PW, T = Cfg::T, R0 = F::R0, NST = F::NST;
    static_assert(NST > 1, "pair pass is for long transforms");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *sm = reinterpret_cast<float4 *>(smem_raw);
    const int tid = threadIdx.x;
    const int c = tid % PW, li = tid / PW;
    const int tile = blockIdx.x % p.n_tiles, lo = blockIdx.x / p.n_tiles, hi = blockIdx.y;

    const float2 *src = p.in + (size_t)hi * p.in_hi + (size_t)lo * p.in_lo + (size_t)tile * TX + 2 * c;
    float2 va[R0], vb[R0];
#pragma unroll
    for (int s = 0; s < R0; ++s) {
        const float4 q = __ldcs(reinterpret_cast<const float4 *>(src + (size_t)(li + s * T) * p.in_row));
        va[s] = make_float2(q.x, q.y); vb[s] = make_float2(q.z, q.w);
    }
    F::stage0(va);
    F::stage0(vb);
    float4 *L = sm + c;
    F::stage0_store2(L, li, va, vb);
    float2 w[R0];
    if constexpr (NST > 2) {
        __syncthreads();
        F::template load_tw<1>(p.tw, li, w);
        F::template stage_load2<1>(L, li, w, va, vb);
        __syncthreads();
        F::template stage_store2<1>(L, li, va, vb);
    }
    if constexpr (NST > 3) {
        __syncthreads();
        F::template load_tw<2>(p.tw, li, w);
        F::template stage_load2<2>(L, li, w, va, vb);
        __syncthreads();
        F::template stage_store2<2>(L, li, va, vb);
    }
    __syncthreads();
    F::template load_tw<NST - 1>(p.tw, li, w);
    F::template stage_load2<NST - 1>(L, li, w, va, vb);
    float2 *dst = p.out + (size_t)hi * p.out_hi + (size_t)lo * p.out_lo + (size_t)tile * TX + 2 * c;
#pragma unroll
    for (int m = 0; m < R0; ++m) {
        const int k = li + T * m;
        const int sl = (k - p.win.lo) & (N - 1);
        if (sl < p.win.W) {
            const float2 a = va[F::out_reg(m)], b = vb[F::out_reg(m)];
            *reinterpret_cast<float4 *>(dst + (size_t)sl * p.out_row) = make_float4(a.x, a.y, b.x, b.y);
        }
    }
}

// Strided pass (z or y axis) for a length that is not a power of two (the paper uses Nz = 63, P:459;
// lateral sizes of any length since DESIGN 3-A14): the definition of Eq. 6 evaluated directly, and only at the window's bins -- the "direct DFT
// at the k_z bins the Ewald pixels need" north_star allows.  A CTA stages a tile of TX columns by N rows
// and the twiddle table in shared memory; thread (c, og) accumulates bins s = og, og + OG, ... of column c.
// The phase index k z mod N is stepped in exact integer arithmetic.  O(W N) per column: meant for the
// short z axes of thin films and for lateral sizes that are not powers of two, not as a general FFT.
// TX columns per tile x OG = 256 / TX bins in flight per column: TX = 32 up to N = 512, TX = 8 beyond (shared memory).
constexpr int DFT_THREADS = 256;
__host__ __device__ constexpr int dft_tx(int N) { return N <= 512 ? 32 : 8; }

template <int TX>
__global__ void __launch_bounds__(DFT_THREADS)
k_coldft(const ColParams p, int N)
{
    pdl_entry();
    constexpr int OG = DFT_THREADS / TX;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *sm = reinterpret_cast<float2 *>(smem_raw);       // [N][TX]
    float2 *tw = sm + (size_t)N * TX;                         // [N]
    const int tid = threadIdx.x, c = tid % TX, og = tid / TX;
    const int tile = blockIdx.x % p.n_tiles, lo = blockIdx.x / p.n_tiles, hi = blockIdx.y;
    const float2 *src = p.in + (size_t)hi * p.in_hi + (size_t)lo * p.in_lo + (size_t)tile * TX + c;
    for (int z = og; z < N; z += OG) sm[z * TX + c] = __ldcs(src + (size_t)z * p.in_row);
    for (int i = tid; i < N; i += DFT_THREADS) tw[i] = p.tw[i];
    __syncthreads();
    float2 *dst = p.out + (size_t)hi * p.out_hi + (size_t)lo * p.out_lo + (size_t)tile * TX + c;
    for (int sl = og; sl < p.win.W; sl += OG) {
        int k = (p.win.lo + sl) % N;
        if (k < 0) k += N;
        // partial sums over 16 terms are added to the total: the rounding error grows like sqrt(16) + sqrt(N / 16)
        // ulps instead of sqrt(N) (N up to 2048)
        float2 tot = make_float2(0.f, 0.f);
        int idx = 0;
        for (int z0 = 0; z0 < N; z0 += 16) {
            float2 a0 = make_float2(0.f, 0.f), a1 = make_float2(0.f, 0.f);
            const int z1 = min(N, z0 + 16);
            int z = z0;
            for (; z + 1 < z1; z += 2) {
                a0 = cfma(sm[z * TX + c], tw[idx], a0);
                idx += k; if (idx >= N) idx -= N;
                a1 = cfma(sm[(z + 1) * TX + c], tw[idx], a1);
                idx += k; if (idx >= N) idx -= N;
            }
            if (z < z1) { a0 = cfma(sm[z * TX + c], tw[idx], a0); idx += k; if (idx >= N) idx -= N; }
            tot = cadd(tot, cadd(a0, a1));
        }
        dst[(size_t)sl * p.out_row] = tot;
    }
}

// ------------------------------------------------------------------------------------------
// x pass of SPECTRAL_BASIS (DESIGN 7.2).  The energy-independent real fields, in material order
//   aligned material:   phi, w = phi S, w dx dx, w dy dy, w dx dy, w dx dz, w dy dz      (7)
//   isotropic material: phi                                                              (1)
// form one global sequence; consecutive fields 2j, 2j+1 are the real and imaginary part of
// complex pack j (the last pack is padded with zeros).  T = N / R0 threads share a row; a thread
// owns the voxels x = li + s T (s < R0), generates their fields in registers, runs the stage-0
// butterfly there, and the remaining stages through a 4-pack shared-memory buffer per row; the
// last stage stores the window [lo, lo + W) of bins straight to out[pack][row][slot].
// sin and cos of a director angle.  CYRSOXS_TRIG = 0: libdevice sincosf (1 ulp; ~50 instructions per call with a
// slow path for large arguments); 1: the special-function unit (MUFU.SIN / MUFU.COS after one multiplication by
// 1/2pi: absolute error ~5e-7 for |x| up to a few pi, 4 instructions).  DESIGN.md 8 derives why 5e-7 on the director
// is far inside the image gates; the parity tests run with whatever is compiled in.
#ifndef CYRSOXS_TRIG
#define CYRSOXS_TRIG 1
#endif
__device__ __forceinline__ void dir_sincos(float x, float *s, float *c)
{
#if CYRSOXS_TRIG == 0
    sincosf(x, s, c);
#else
    *s = __sinf(x); *c = __cosf(x);
#endif
}

// x pass of SPECTRAL_BASIS for a row length that is not a power of two (DESIGN 3-A14): the definition
// of Eq. 6 evaluated directly, and only at the window's bins.  One CTA per row; per pack the two real fields of the row are
// generated into shared memory (kind / material tables of the basis plan), then thread `sl` accumulates bin (lo + sl) mod N.
// O(W N) per row and pack: a functional path for modest sizes, not a tuned FFT (measured, DESIGN 12.4: a 1000 x 600 x 1
// film 2.4 ms, a 1000 x 1000 x 64 volume 203 ms against 0.6 ms for the 1024-point FFT pass).
constexpr int XDFT_THREADS = 256;

__device__ __forceinline__ float basis_field(const MorphPtrs &mp, int kind, int m, size_t vox)
{
    if (kind == BK_NONE) return 0.f;
    const float ph = __ldg(mp.phi[m] + vox);
    if (kind == BK_PHI) return ph;
    const float w = ph * __ldg(mp.S[m] + vox);
    if (kind == BK_W) return w;
    float st, ct, sp, cp;
    dir_sincos(__ldg(mp.theta[m] + vox), &st, &ct);
    dir_sincos(__ldg(mp.psi[m] + vox), &sp, &cp);
    const float dx = cp * st, dy = sp * st, dz = ct;
    switch (kind) {
    case BK_XX: return (w * dx) * dx;
    case BK_YY: return (w * dy) * dy;
    case BK_XY: return (w * dx) * dy;
    case BK_XZ: return (w * dx) * dz;
    default: return (w * dy) * dz;        // BK_YZ
    }
}

__global__ void __launch_bounds__(XDFT_THREADS)
k_xdft(const __grid_constant__ MorphPtrs mp, const int *__restrict__ kind, const int *__restrict__ mat_of, int mat_base, int n_pack,
       float2 *__restrict__ out, int rows_total, size_t fstride, Window wx, int pitch, const float2 *__restrict__ tw_g, int N)
{
    pdl_entry();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *f = reinterpret_cast<float2 *>(smem_raw);        // [N] the pack's row
    float2 *tw = f + N;                                       // [N] exp(-2 pi i t / N)
    const int tid = threadIdx.x, row = blockIdx.x;
    if (row >= rows_total) return;
    for (int i = tid; i < N; i += XDFT_THREADS) tw[i] = tw_g[i];
    const size_t vox0 = (size_t)row * N;
    for (int pk = 0; pk < n_pack; ++pk) {
        __syncthreads();                                     // the previous pack's sums are done with f (and tw is loaded)
        const int ka = kind[2 * pk], kb = kind[2 * pk + 1], ma = mat_of[2 * pk] - mat_base, mb = mat_of[2 * pk + 1] - mat_base;
        for (int x = tid; x < N; x += XDFT_THREADS) f[x] = make_float2(basis_field(mp, ka, ma, vox0 + x), basis_field(mp, kb, mb, vox0 + x));
        __syncthreads();
        float2 *o = out + (size_t)pk * fstride + (size_t)row * pitch;
        for (int sl = tid; sl < pitch; sl += XDFT_THREADS) {
            float2 tot = make_float2(0.f, 0.f);
            if (sl < wx.W) {
                int k = (wx.lo + sl) % N;
                if (k < 0) k += N;
                int idx = 0;
                for (int x0 = 0; x0 < N; x0 += 16) {         // partial sums over 16 terms, see k_coldft
                    float2 a0 = make_float2(0.f, 0.f), a1 = make_float2(0.f, 0.f);
                    const int x1 = min(N, x0 + 16);
                    int x = x0;
                    for (; x + 1 < x1; x += 2) {
                        a0 = cfma(f[x], tw[idx], a0);
                        idx += k; if (idx >= N) idx -= N;
                        a1 = cfma(f[x + 1], tw[idx], a1);
                        idx += k; if (idx >= N) idx -= N;
                    }
                    if (x < x1) { a0 = cfma(f[x], tw[idx], a0); idx += k; if (idx >= N) idx -= N; }
                    tot = cadd(tot, cadd(a0, a1));
                }
            }
            o[sl] = tot;                                     // slots [W, pitch) are the row's zero padding
        }
    }
}

constexpr int XB2_PB = 4;       // packs buffered per row between flushes
static_assert(XB2_PB >= 4, "an aligned material emits up to 4 packs between flush checks");
// CTAs per SM the register allocation aims at: 3 (80 registers, a few spilled values) measured 9-12 % faster
// than 2 (126 registers) on CFG2, CFG3 and CFG5 -- the kernel is latency bound at 16 warps per SM.
constexpr int XB2_MINB = 3;

template <int LOGN> struct XB2Cfg {
    static constexpr int N = 1 << LOGN;
    using F = RegFft<LOGN, RowMap>;
    static constexpr int T = F::T, R0 = F::R0;
    static constexpr int ROWS = T >= 256 ? 1 : 256 / T;
    static constexpr int THREADS = ROWS * T;
    static constexpr size_t SMEM = F::NST > 1 ? sizeof(float2) * (size_t)ROWS * XB2_PB * N : 0;
};

template <int LOGN>
__global__ void __launch_bounds__(XB2Cfg<LOGN>::THREADS, XB2_MINB)
k_xbasis2(const __grid_constant__ MorphPtrs mp, float2 *__restrict__ out, int rows_total, size_t fstride, Window wx, int pitch,
          const float2 *__restrict__ tw)
{
    pdl_entry();
    using Cfg = XB2Cfg<LOGN>;
    using F = typename Cfg::F;
    constexpr int N = Cfg::N, T = Cfg::T, R0 = Cfg::R0, NST = F::NST, THREADS = Cfg::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int g = tid / T, li = tid % T;
    const int row = blockIdx.x * Cfg::ROWS + g;
    const bool row_ok = row < rows_total;
    const int rowc = row_ok ? row : rows_total - 1;
    float2 *Lrow = reinterpret_cast<float2 *>(smem_raw) + (size_t)g * (XB2_PB * N);
    const size_t vox0 = (size_t)rowc * N + li;
    float2 *orow = out + (size_t)rowc * pitch;

    float carry[R0];
    bool has_carry = false;
    int nbuf = 0, pack_out = 0;

    // The thread's outputs are the bins k = li + T m; bin k goes to slot (k - lo) mod N when that is inside the row
    // (slots [W, pitch) are the row's zero padding).  Slot offsets, a store mask and a zero mask are worked out once.
    int soff[R0];
    unsigned int st_mask = 0, zero_mask = 0;
#pragma unroll
    for (int m = 0; m < R0; ++m) {
        const int sl = (li + T * m - wx.lo) & (N - 1);
        soff[m] = sl;
        if (sl < pitch && row_ok) st_mask |= 1u << m;
        if (sl >= wx.W) zero_mask |= 1u << m;
    }
    auto store_global = [&](int pack, const float2 (&v)[R0]) {
        float2 *o = orow + (size_t)pack * fstride;
#pragma unroll
        for (int m = 0; m < R0; ++m)
            if (st_mask >> m & 1u) o[soff[m]] = (zero_mask >> m & 1u) ? make_float2(0.f, 0.f) : v[F::out_reg(m)];
        if (N < 32) {
            for (int sl = N + li; sl < pitch; sl += T)
                if (row_ok) o[sl] = make_float2(0.f, 0.f);
        }
    };
    // one complex pack from two real fields given as generators fa(s), fb(s) of the thread's voxel s:
    // the products are formed here, right before the stage-0 butterfly, so only w, d and phi stay live
    auto emit = [&](auto fa, auto fb) {
        float2 v[R0];
#pragma unroll
        for (int s = 0; s < R0; ++s) v[s] = make_float2(fa(s), fb(s));
        F::stage0(v);
        if constexpr (NST > 1) { F::stage0_store(Lrow + nbuf * N, li, v); ++nbuf; }
        else { store_global(pack_out, v); ++pack_out; }
    };
    auto flush = [&]() {
        if constexpr (NST > 1) {
            float2 w[R0], v[R0];
            if constexpr (NST > 2) {
                group_sync<T, THREADS>(g);
                F::template load_tw<1>(tw, li, w);
                for (int pk = 0; pk < nbuf; ++pk) {
                    F::template stage_load<1>(Lrow + pk * N, li, w, v);
                    group_sync<T, THREADS>(g);
                    F::template stage_store<1>(Lrow + pk * N, li, v);
                }
            }
            if constexpr (NST > 3) {
                group_sync<T, THREADS>(g);
                F::template load_tw<2>(tw, li, w);
                for (int pk = 0; pk < nbuf; ++pk) {
                    F::template stage_load<2>(Lrow + pk * N, li, w, v);
                    group_sync<T, THREADS>(g);
                    F::template stage_store<2>(Lrow + pk * N, li, v);
                }
            }
            group_sync<T, THREADS>(g);
            F::template load_tw<NST - 1>(tw, li, w);
            for (int pk = 0; pk < nbuf; ++pk) {
                F::template stage_load<NST - 1>(Lrow + pk * N, li, w, v);
                store_global(pack_out + pk, v);
            }
            group_sync<T, THREADS>(g);          // the buffer is reused by the next stage-0 stores
            pack_out += nbuf;
            nbuf = 0;
        }
    };

    for (int m = 0; m < mp.n_mat; ++m) {
        const bool aligned = mp.S[m] != nullptr;
        if (nbuf + (aligned ? 4 : 1) > XB2_PB) flush();
        float ph[R0];
#pragma unroll
        for (int s = 0; s < R0; ++s) ph[s] = __ldcs(mp.phi[m] + vox0 + (size_t)s * T);
        if (aligned) {
            float S_[R0], th[R0], ps[R0];
#pragma unroll
            for (int s = 0; s < R0; ++s) {
                S_[s] = __ldcs(mp.S[m] + vox0 + (size_t)s * T);
                th[s] = __ldcs(mp.theta[m] + vox0 + (size_t)s * T);
                ps[s] = __ldcs(mp.psi[m] + vox0 + (size_t)s * T);
            }
            float w[R0], dx[R0], dy[R0], dz[R0];
#pragma unroll
            for (int s = 0; s < R0; ++s) {
                w[s] = ph[s] * S_[s];
                float st, ct, sp, cp;
                dir_sincos(th[s], &st, &ct);
                dir_sincos(ps[s], &sp, &cp);
                dx[s] = cp * st; dy[s] = sp * st; dz[s] = ct;
            }
            auto f_ph = [&](int s) { return ph[s]; };
            auto f_w = [&](int s) { return w[s]; };
            auto f_xx = [&](int s) { return (w[s] * dx[s]) * dx[s]; };
            auto f_yy = [&](int s) { return (w[s] * dy[s]) * dy[s]; };
            auto f_xy = [&](int s) { return (w[s] * dx[s]) * dy[s]; };
            auto f_xz = [&](int s) { return (w[s] * dx[s]) * dz[s]; };
            auto f_yz = [&](int s) { return (w[s] * dy[s]) * dz[s]; };
            if (has_carry) {
                emit([&](int s) { return carry[s]; }, f_ph); emit(f_w, f_xx); emit(f_yy, f_xy); emit(f_xz, f_yz);
                has_carry = false;
            } else {
                emit(f_ph, f_w); emit(f_xx, f_yy); emit(f_xy, f_xz);
#pragma unroll
                for (int s = 0; s < R0; ++s) carry[s] = f_yz(s);
                has_carry = true;
            }
        } else {
            if (has_carry) { emit([&](int s) { return carry[s]; }, [&](int s) { return ph[s]; }); has_carry = false; }
            else {
#pragma unroll
                for (int s = 0; s < R0; ++s) carry[s] = ph[s];
                has_carry = true;
            }
        }
    }
    if (has_carry) {
        if (nbuf + 1 > XB2_PB) flush();
        emit([&](int s) { return carry[s]; }, [](int) { return 0.f; });
    }
    flush();
}

// ------------------------------------------------------------------------------------------
// x pass of SPECTRAL_BASIS, second generation (N = 64 .. 2048; shorter rows keep k_xbasis2).  Same fields, same
// pack order and same output layout as k_xbasis2; what differs is how a row is transformed (fft2.cuh):
//   * the packs buffered in shared memory go through the later stages two at a time: 16 values per thread, one
//     barrier per pair and stage, radix 16 in the middle of 1024- and 2048-point rows (2 trips through shared
//     memory instead of 3; 128 points: 1 instead of 2);
//   * per-stage twiddle tables read with unit stride;
//   * the window store works from one precomputed slot per thread (k0) and compile-time offsets;
//   * sin / cos of the director angles on the special-function unit (dir_sincos);
//   * the next material's rows are prefetched into L2 while the current one is transformed.
constexpr int XB3_PB = 4;
// CTA shape (measured on B200, CFG3 / CFG5 x pass in ms): 256 threads at 128 registers (2 CTAs/SM) 1.24 / 8.8; 128
// threads at 128 registers (4 CTAs/SM) 1.13 / 8.0; 128 threads at 96 registers (5 CTAs/SM, a few spills) 1.21 / 7.7;
// 80 registers (heavy spills) 1.5 / 9.3-11.  The kernel is latency bound (ncu: issue slots 52 % busy at 16 warps per
// SM), so small CTAs -- finer-grained refill of the SM -- and the fifth CTA pay at 1024 points.
#ifndef CYRSOXS_XB3_CTA
#define CYRSOXS_XB3_CTA 128
#endif

template <int LOGN, int CTA> struct XB3CfgT {
    static constexpr int N = 1 << LOGN;
    using F = Fft2<LOGN>;
    static constexpr int T = F::T;
    static constexpr int ROWS = T >= CTA ? 1 : CTA / T;
    static constexpr int THREADS = ROWS * T;
#ifdef CYRSOXS_XB3_MINB
    static constexpr int MINB = CYRSOXS_XB3_MINB;
#else
    static constexpr int MINB = THREADS > 128 ? 2 : (LOGN == 10 ? 5 : 4);
#endif
    static constexpr int LSTRIDE = PadMap::line(N) + (N <= 128 ? 8 : 0);   // line stride: keeps the two lines of a split
    static constexpr int RSTRIDE = XB3_PB * LSTRIDE + (N == 64 ? 8 : 0);    // stage / two rows of a half-warp on distinct banks
    static constexpr size_t SMEM = sizeof(float2) * (size_t)ROWS * RSTRIDE;
};
template <int LOGN> using XB3Cfg = XB3CfgT<LOGN, CYRSOXS_XB3_CTA>;

// The work of one CTA of the x pass: rows [row_first, row_first + ROWS) of a block of rows_total rows whose first voxel is
// vox_off (into every morphology array); pack p of row r goes to out[p fstride + r pitch + slot].
template <int LOGN, int CTA>
__device__ __forceinline__ void xbasis3_rows(const MorphPtrs &mp, size_t vox_off, float2 *__restrict__ out, int row_first, int rows_total,
                                             size_t fstride, const Window &wx, int pitch, const float2 *__restrict__ tws, int rows_ahead,
                                             unsigned char *smem_raw, int tid)
{
    using Cfg = XB3CfgT<LOGN, CTA>;
    using F = typename Cfg::F;
    using Map = PadMap;
    constexpr int N = Cfg::N, T = Cfg::T, NST = F::NST, THREADS = Cfg::THREADS, LS = Cfg::LSTRIDE;
    const int g = tid / T, li = tid % T;
    const int row = row_first + g;
    const bool row_ok = row < rows_total;
    const int rowc = row_ok ? row : rows_total - 1;
    float2 *Lrow = reinterpret_cast<float2 *>(smem_raw) + (size_t)g * Cfg::RSTRIDE;
    const size_t vox0 = vox_off + (size_t)rowc * N + li;
    float2 *orow = out + (size_t)rowc * pitch;

    float carry[8];
    bool has_carry = false;
    int nbuf = 0, pack_out = 0;
    const int lo = wx.lo, W = wx.W;

    // bin k of pack `pack` goes to slot (k - lo) mod N if that is inside the row; slots [W, pitch) are zero padding
    auto store_bin = [&](int pack, int k, float2 val) {
        const int sl = (k - lo) & (N - 1);
        if (sl < pitch && row_ok) orow[(size_t)pack * fstride + sl] = sl < W ? val : make_float2(0.f, 0.f);
    };
    auto emit = [&](auto fa, auto fb) {
        float2 v[8];
#pragma unroll
        for (int s = 0; s < 8; ++s) v[s] = make_float2(fa(s), fb(s));
        F::stage0(v);
        F::template stage0_store<Map>(Lrow + nbuf * LS, li, v);
        ++nbuf;
    };
    auto flush = [&]() {
        float2 w[8], v[16];
        if constexpr (NST > 2) {
            group_sync<T, THREADS>(g);
            F::template load_tw<1>(tws, li, w);
            for (int pk = 0; pk < nbuf; pk += 2) {
                float2 *LA = Lrow + pk * LS, *LB = LA + LS;
                const bool hasB = pk + 1 < nbuf;
                F::template stage_load<1, Map>(LA, LB, hasB, li, w, v);
                group_sync<T, THREADS>(g);
                F::template stage_store<1, Map>(LA, LB, hasB, li, v);
            }
        }
        group_sync<T, THREADS>(g);
        F::template load_tw<NST - 1>(tws, li, w);
        for (int pk = 0; pk < nbuf; pk += 2) {
            float2 *LA = Lrow + pk * LS, *LB = LA + LS;
            const bool hasB = pk + 1 < nbuf;
            F::template stage_load<NST - 1, Map>(LA, LB, hasB, li, w, v);
            const int p0 = pack_out + pk;
            F::for_each_output(hasB, li, v, [&](int line, int k, float2 val) { store_bin(p0 + line, k, val); });
        }
        group_sync<T, THREADS>(g);          // the buffer is reused by the next stage-0 stores
        pack_out += nbuf;
        nbuf = 0;
    };
    // one 128-byte line per lane: the T threads of a row cover its N floats with N / 32 prefetches per array
    auto prefetch_row_of = [&](const float *a, int r) {
        if (li < N / 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(a + vox_off + (size_t)r * N + li * 32));
    };
    auto prefetch_row = [&](const float *a) { prefetch_row_of(a, rowc); };
    // the first material of the rows a later CTA will start with (rows_ahead ~ the rows in flight on the whole GPU):
    // that CTA's first loads then hit L2 instead of exposing the DRAM latency at the start of its short life
    if (row + rows_ahead < rows_total) {
        prefetch_row_of(mp.phi[0], row + rows_ahead);
        if (mp.S[0]) { prefetch_row_of(mp.S[0], row + rows_ahead); prefetch_row_of(mp.theta[0], row + rows_ahead); prefetch_row_of(mp.psi[0], row + rows_ahead); }
    }

    for (int m = 0; m < mp.n_mat; ++m) {
        const bool aligned = mp.S[m] != nullptr;
        if (nbuf + (aligned ? 4 : 1) > XB3_PB) flush();
        float ph[8];
#pragma unroll
        for (int s = 0; s < 8; ++s) ph[s] = __ldcs(mp.phi[m] + vox0 + (size_t)s * T);
        if (m + 1 < mp.n_mat) {
            prefetch_row(mp.phi[m + 1]);
            if (mp.S[m + 1]) { prefetch_row(mp.S[m + 1]); prefetch_row(mp.theta[m + 1]); prefetch_row(mp.psi[m + 1]); }
        }
        if (aligned) {
            float S_[8], th[8], ps[8];
#pragma unroll
            for (int s = 0; s < 8; ++s) {
                S_[s] = __ldcs(mp.S[m] + vox0 + (size_t)s * T);
                th[s] = __ldcs(mp.theta[m] + vox0 + (size_t)s * T);
                ps[s] = __ldcs(mp.psi[m] + vox0 + (size_t)s * T);
            }
            float w[8], dx[8], dy[8], dz[8];
#pragma unroll
            for (int s = 0; s < 8; ++s) {
                w[s] = ph[s] * S_[s];
                float st, ct, sp, cp;
                dir_sincos(th[s], &st, &ct);
                dir_sincos(ps[s], &sp, &cp);
                dx[s] = cp * st; dy[s] = sp * st; dz[s] = ct;
            }
            auto f_ph = [&](int s) { return ph[s]; };
            auto f_w = [&](int s) { return w[s]; };
            auto f_xx = [&](int s) { return (w[s] * dx[s]) * dx[s]; };
            auto f_yy = [&](int s) { return (w[s] * dy[s]) * dy[s]; };
            auto f_xy = [&](int s) { return (w[s] * dx[s]) * dy[s]; };
            auto f_xz = [&](int s) { return (w[s] * dx[s]) * dz[s]; };
            auto f_yz = [&](int s) { return (w[s] * dy[s]) * dz[s]; };
            if (has_carry) {
                emit([&](int s) { return carry[s]; }, f_ph); emit(f_w, f_xx); emit(f_yy, f_xy); emit(f_xz, f_yz);
                has_carry = false;
            } else {
                emit(f_ph, f_w); emit(f_xx, f_yy); emit(f_xy, f_xz);
#pragma unroll
                for (int s = 0; s < 8; ++s) carry[s] = f_yz(s);
                has_carry = true;
            }
        } else {
            if (has_carry) { emit([&](int s) { return carry[s]; }, [&](int s) { return ph[s]; }); has_carry = false; }
            else {
#pragma unroll
                for (int s = 0; s < 8; ++s) carry[s] = ph[s];
                has_carry = true;
            }
        }
    }
    if (has_carry) {
        if (nbuf + 1 > XB3_PB) flush();
        emit([&](int s) { return carry[s]; }, [](int) { return 0.f; });
    }
    flush();
}

template <int LOGN>
__global__ void __launch_bounds__(XB3Cfg<LOGN>::THREADS, XB3Cfg<LOGN>::MINB)
k_xbasis3(const __grid_constant__ MorphPtrs mp, float2 *__restrict__ out, int rows_total, size_t fstride, Window wx, int pitch,
          const float2 *__restrict__ tws, int rows_ahead)
{
    pdl_entry();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    xbasis3_rows<LOGN, CYRSOXS_XB3_CTA>(mp, 0, out, blockIdx.x * XB3Cfg<LOGN>::ROWS, rows_total, fstride, wx, pitch, tws, rows_ahead, smem_raw, threadIdx.x);
}

} // namespace cyr
