// fft_core.cuh -- shared-memory Stockham FFT building blocks (forward, exp(-2 pi i jk/N),
// unnormalised: Eq. 6).  Lengths 2^1 .. 2^11, radix 8/4/2 butterflies held in
// registers, twiddles from a table computed in double on the host and rounded once.
//
// One stage (radix R, Ns = product of the radices already done), butterfly j in [0, N/R):
//   in   x[j + s N/R],                     s = 0..R-1
//   tw   exp(-2 pi i s (j mod Ns) / (Ns R))
//   out  y[(j / Ns) Ns R + (j mod Ns) + t Ns], t = 0..R-1      (autosort: natural order at the end)
// Stages run in place: every thread reads its butterflies into registers, the block
// synchronises, then writes.
//
// Shared-memory layout ("accessor"):
//   RowAcc  a line is contiguous; re and im in separate float arrays, index i stored at
//           i + (i >> 5) (one pad word per 32) so that the stride-R writes of the early stages
//           and the unit-stride reads are both bank-conflict free.  Used by the x pass, where
//           lanes run along the transform axis.
// (the strided z and y passes keep their lines in registers and in the layouts of fft_reg.cuh)
#pragma once
#include <cuda_runtime.h>

namespace cyr {

// Packed fp32 arithmetic (sm_100a: add/sub/mul/fma.rn.f32x2 -> FADD2 / FMUL2 / FFMA2).  One instruction does
// the real and the imaginary part of a complex value, and ptxas folds the swaps, sign changes and scalar
// broadcasts of the operands into the instruction's operand modifiers (R.F32x2.LO_HI.NP, R.F32), so a complex
// add is 1 issue slot instead of 2 and a complex multiply 2 instead of 4.  The FMA pipe does the same number of
// lane operations either way (measured: 116-122 lane-ops/clk/SM for FFMA and FFMA2 alike); what is saved is
// issue slots, which the loads, stores and address arithmetic of an FFT pass need.  Every operation is
// individually rounded (.rn), i.e. identical results to the scalar form.
namespace pk {
__device__ __forceinline__ float2 add(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 sub(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 mul(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mul.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 fma(float2 a, float2 b, float2 c)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mov.b64 rc, {%6,%7}; fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}
} // namespace pk

// v * w: (v.x w.x - v.y w.y, v.y w.x + v.x w.y) = v (w.x, w.x) + (-v.y, v.x)(w.y, w.y): FMUL2 + FFMA2
__device__ __forceinline__ float2 cmul(float2 v, float2 w)
{
    return pk::fma(make_float2(-v.y, v.x), make_float2(w.y, w.y), pk::mul(v, make_float2(w.x, w.x)));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return pk::add(a, b); }
// a * b + c
__device__ __forceinline__ float2 cfma(float2 a, float2 b, float2 c)
{
    return pk::fma(make_float2(-a.y, a.x), make_float2(b.y, b.y), pk::fma(a, make_float2(b.x, b.x), c));
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return pk::sub(a, b); }
// multiply by -i (forward-transform quarter turn): a swap and a sign, folded into the consumer's operand modifiers
__device__ __forceinline__ float2 cmul_mi(float2 a) { return make_float2(a.y, -a.x); }

template <int R> struct Dft;

template <> struct Dft<2> {
    __device__ __forceinline__ static void run(float2 *v)
    {
        float2 a = v[0], b = v[1];
        v[0] = cadd(a, b); v[1] = csub(a, b);
    }
};

template <> struct Dft<4> {
    __device__ __forceinline__ static void run(float2 *v)
    {
        float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        float2 t2 = cadd(v[1], v[3]), t3 = cmul_mi(csub(v[1], v[3]));
        v[0] = cadd(t0, t2); v[1] = cadd(t1, t3); v[2] = csub(t0, t2); v[3] = csub(t1, t3);
    }
};

template <> struct Dft<8> {
    // 8 = 2 x 4 decimation in frequency: b_k = v_k + v_{k+4}, c_k = (v_k - v_{k+4}) w8^k,
    // Y[2m] = DFT4(b)[m], Y[2m+1] = DFT4(c)[m].
    __device__ __forceinline__ static void run(float2 *v)
    {
        const float h = 0.70710678118654752440f;
        float2 b[4], c[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { b[k] = cadd(v[k], v[k + 4]); c[k] = csub(v[k], v[k + 4]); }
        c[1] = pk::mul(make_float2(h, h), pk::add(c[1], make_float2(c[1].y, -c[1].x)));      // * (1 - i)/sqrt2
        c[2] = cmul_mi(c[2]);                                                                  // * -i
        c[3] = pk::mul(make_float2(-h, -h), pk::add(c[3], make_float2(-c[3].y, c[3].x)));    // * (-1 - i)/sqrt2
        Dft<4>::run(b); Dft<4>::run(c);
#pragma unroll
        for (int m = 0; m < 4; ++m) { v[2 * m] = b[m]; v[2 * m + 1] = c[m]; }
    }
};

// ---------------------------------------------------------------------------- accessors

template <int N> struct RowLayout {
    // first-stage input layout written by the field generator: element x of a line sits at
    // (x & 3) * QSTRIDE + (x >> 2): the four voxels a thread produces go to four quarter
    // blocks, lanes contiguous inside each (conflict-free stores), and the quarter stride is
    // 8 (mod 32) so that the first stage's unit-stride reads are conflict-free too.
    static constexpr bool PERMUTED_INPUT = (N >= 32);
    static constexpr int QSTRIDE = N / 4 + 8;
    static constexpr int PADDED = N + (N >> 5);
    static constexpr int LS_RAW = PERMUTED_INPUT ? (4 * QSTRIDE > PADDED ? 4 * QSTRIDE : PADDED) : PADDED;
    static constexpr int LS = LS_RAW | 1;           // odd line stride: lanes spanning lines hit distinct banks
    __device__ __forceinline__ static int input_pos(int x)
    {
        return PERMUTED_INPUT ? (x & 3) * QSTRIDE + (x >> 2) : x + (x >> 5);
    }
    __device__ __forceinline__ static int pos(int i) { return i + (i >> 5); }
};

template <int N> struct RowAcc {
    float *re, *im;
    using L = RowLayout<N>;
    template <int NB> __device__ __forceinline__ static void split(int w, int, int &line, int &j)
    {
        line = w / NB; j = w % NB;
    }
    __device__ __forceinline__ float2 load(int line, int i) const
    {
        int p = line * L::LS + L::pos(i);
        return make_float2(re[p], im[p]);
    }
    __device__ __forceinline__ float2 load_input(int line, int i) const
    {
        int p = line * L::LS + L::input_pos(i);
        return make_float2(re[p], im[p]);
    }
    __device__ __forceinline__ void store(int line, int i, float2 v) const
    {
        int p = line * L::LS + L::pos(i);
        re[p] = v.x; im[p] = v.y;
    }
};

// ---------------------------------------------------------------------------- one stage

template <int N, int R, int NS, int NLINES_MAX, int THREADS, bool FIRST, class Acc>
__device__ __forceinline__ void fft_stage(const Acc &acc, int nlines, const float2 *__restrict__ tw, int tid)
{
    constexpr int NB = N / R;
    constexpr int TOTAL_MAX = NLINES_MAX * NB;
    constexpr int BPT = (TOTAL_MAX + THREADS - 1) / THREADS;
    const int total = nlines * NB;
    float2 v[BPT][R];
#pragma unroll
    for (int b = 0; b < BPT; ++b) {
        int w = tid + b * THREADS;
        if (w < total) {
            int line, j;
            Acc::template split<NB>(w, nlines, line, j);
#pragma unroll
            for (int s = 0; s < R; ++s)
                v[b][s] = FIRST ? acc.load_input(line, j + s * NB) : acc.load(line, j + s * NB);
            if (NS > 1) {
                const int t0 = (j & (NS - 1)) * (N / (NS * R));
#pragma unroll
                for (int s = 1; s < R; ++s) v[b][s] = cmul(v[b][s], tw[s * t0]);
            }
            Dft<R>::run(v[b]);
        }
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < BPT; ++b) {
        int w = tid + b * THREADS;
        if (w < total) {
            int line, j;
            Acc::template split<NB>(w, nlines, line, j);
            const int o = (j / NS) * (NS * R) + (j & (NS - 1));
#pragma unroll
            for (int t = 0; t < R; ++t) acc.store(line, o + t * NS, v[b][t]);
        }
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------- whole transform

// Radix schedule for 2^LOGN: as many 8s as possible, remainder as 4s / one 2, e.g.
// 128 = 8.4.4, 256 = 8.8.4, 512 = 8.8.8, 1024 = 8.8.4.4, 2048 = 8.8.8.4.
template <int LOGN> struct Radices {
    static constexpr int REM = LOGN % 3;
    static constexpr int N8 = (REM == 1 && LOGN >= 4) ? LOGN / 3 - 1 : LOGN / 3;
    static constexpr int LEFT = LOGN - 3 * N8;       // 0, 1, 2 or 4 bits left
    static constexpr int N4 = LEFT / 2;
    static constexpr int N2 = LEFT % 2;
};

template <int LOGN, int NLINES_MAX, int THREADS, class Acc, int STAGE = 0, int LOGNS = 0>
struct FftRun {
    using Rd = Radices<LOGN>;
    static constexpr int N = 1 << LOGN;
    static constexpr int R = STAGE < Rd::N8 ? 8 : (STAGE < Rd::N8 + Rd::N4 ? 4 : 2);
    static constexpr int LOGR = R == 8 ? 3 : (R == 4 ? 2 : 1);
    __device__ __forceinline__ static void run(const Acc &acc, int nlines, const float2 *tw, int tid)
    {
        if constexpr (LOGNS < LOGN) {
            fft_stage<N, R, (1 << LOGNS), NLINES_MAX, THREADS, (STAGE == 0), Acc>(acc, nlines, tw, tid);
            FftRun<LOGN, NLINES_MAX, THREADS, Acc, STAGE + 1, LOGNS + LOGR>::run(acc, nlines, tw, tid);
        }
    }
};

// Transforms `nlines` lines of length 2^LOGN held in shared memory through `acc`.
// All THREADS threads of the block must call it; data must be visible (caller syncs before).
template <int LOGN, int NLINES_MAX, int THREADS, class Acc>
__device__ __forceinline__ void fft_lines(const Acc &acc, int nlines, const float2 *tw, int tid)
{
    FftRun<LOGN, NLINES_MAX, THREADS, Acc>::run(acc, nlines, tw, tid);
}

} // namespace cyr
