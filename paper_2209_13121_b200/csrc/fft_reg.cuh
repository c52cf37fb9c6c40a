// fft_reg.cuh -- register-first / register-last Stockham FFT (forward, exp(-2 pi i jk/N),
// unnormalised: Eq. 6) for lengths 2^1 .. 2^11.
//
// A line of length N = R0 R1 .. is transformed by T = N / R0 threads; every thread keeps R0
// complex values in registers for the whole transform:
//   stage 0   the thread's inputs x[li + s T] (s < R0) are ALREADY in registers (loaded from
//             global memory or generated there); one radix-R0 butterfly; the results go to
//             shared memory at the autosort positions li R0 + t;
//   middle    B = R0 / R butterflies of radix R per thread: read x[j + s N/R], j = li + b T,
//             multiply by exp(-2 pi i s (j mod Ns) / (Ns R)), butterfly, write
//             y[(j / Ns) Ns R + (j mod Ns) + t Ns]   (in place: the group synchronises between
//             the reads and the writes);
//   last      same reads; the outputs k = li + T m (m < R0) STAY in registers and the caller
//             stores them straight to global memory (value of bin k is v[(m % B) R + m / B]).
// So a transform costs (stages - 1) shared-memory round trips instead of (stages + 1), with
// 64-bit accesses.  Twiddles come from a table exp(-2 pi i t / N) computed in double on the
// host and rounded once.
#pragma once
#include <cuda_runtime.h>
#include "fft_core.cuh"

namespace cyr {

template <> struct Dft<1> {
    __device__ __forceinline__ static void run(float2 *) {}
};

// radix schedule: first radix R0 is the largest, later radices divide it
template <int LOGN> struct RSched;
template <> struct RSched<1> { static constexpr int NST = 1; static constexpr int R[4] = {2, 1, 1, 1}; };
template <> struct RSched<2> { static constexpr int NST = 1; static constexpr int R[4] = {4, 1, 1, 1}; };
template <> struct RSched<3> { static constexpr int NST = 1; static constexpr int R[4] = {8, 1, 1, 1}; };
template <> struct RSched<4> { static constexpr int NST = 2; static constexpr int R[4] = {4, 4, 1, 1}; };
template <> struct RSched<5> { static constexpr int NST = 2; static constexpr int R[4] = {8, 4, 1, 1}; };
template <> struct RSched<6> { static constexpr int NST = 2; static constexpr int R[4] = {8, 8, 1, 1}; };
template <> struct RSched<7> { static constexpr int NST = 3; static constexpr int R[4] = {8, 4, 4, 1}; };
template <> struct RSched<8> { static constexpr int NST = 3; static constexpr int R[4] = {8, 8, 4, 1}; };
template <> struct RSched<9> { static constexpr int NST = 3; static constexpr int R[4] = {8, 8, 8, 1}; };
template <> struct RSched<10> { static constexpr int NST = 4; static constexpr int R[4] = {8, 8, 4, 4}; };
template <> struct RSched<11> { static constexpr int NST = 4; static constexpr int R[4] = {8, 8, 8, 4}; };

// Shared-memory addressing of element i of a line.
//   RowMap   the line is contiguous (float2 L[N]); i is XOR-swizzled with bits 3..6 so that the
//            stride-R0 writes of stage 0, the stride-Ns writes of the later stages and the
//            unit-stride reads are all bank-conflict free per half-warp (64-bit accesses).
//   ColMap   TX independent lines side by side, element i of line c at (i' TX + c): lanes run
//            across the columns.  For TX = 8 two butterflies share a half-warp, so bit 0 of i is
//            flipped for odd i >> 3; for TX = 4 bits 0..1 are XORed with bits 3..4.
struct RowMap {
    __device__ __forceinline__ static int at(int i) { return i ^ ((i >> 3) & 15); }
    // at(i + c) from a = at(i) for a compile-time offset c that is a multiple of 64: the swizzle reads
    // bits 3..6 and writes bits 0..3, so a multiple of 128 commutes with it and an odd multiple of 64
    // flips bit 6, i.e. toggles bit 3 of the mask.  Saves the shift/and/xor per access.
    static constexpr bool kSwizzled = true;
    __device__ __forceinline__ static int shifted(int a, int c) { return ((c & 64) ? (a ^ 8) : a) + c; }
};
template <int TX> struct ColMap {
    static constexpr bool kSwizzled = false;
    __device__ __forceinline__ static int at(int i)
    {
        if (TX >= 16) return i * TX;
        if (TX == 8) return (i ^ ((i >> 3) & 1)) * TX;
        return (i ^ ((i >> 3) & 3)) * TX;
    }
};

// Pairs of lines as float4: PW pairs side by side, element i of pair c at (i PW + c).  With PW = 8 a
// quarter-warp (one 128-bit wavefront) covers one full 128-byte row, so no swizzle is needed.
template <int PW> struct PairMap {
    static constexpr bool kSwizzled = false;
    __device__ __forceinline__ static int at(int i) { return i * PW; }
};

template <int LOGN, class Map> struct RegFft {
    using S = RSched<LOGN>;
    static constexpr int N = 1 << LOGN;
    static constexpr int NST = S::NST;
    static constexpr int R0 = S::R[0];
    static constexpr int T = N / R0;               // threads per line

    __host__ __device__ static constexpr int ns_of(int stage)
    {
        int ns = 1;
        for (int s = 0; s < stage; ++s) ns *= S::R[s];
        return ns;
    }

    // stage 0: butterfly on the register inputs (v[s] = x[li + s T]); v then holds y[li R0 + t].
    __device__ __forceinline__ static void stage0(float2 (&v)[R0]) { Dft<R0>::run(v); }

    // writes the stage-0 results to shared memory (only when NST > 1)
    __device__ __forceinline__ static void stage0_store(float2 *L, int li, const float2 (&v)[R0])
    {
#pragma unroll
        for (int t = 0; t < R0; ++t) L[Map::at(li * R0 + t)] = v[t];
    }

    // twiddles of stage ST (>= 1) for this thread: w[b R + s], s >= 1
    template <int ST>
    __device__ __forceinline__ static void load_tw(const float2 *__restrict__ tw, int li, float2 (&w)[R0])
    {
        constexpr int R = S::R[ST], B = R0 / R, NS = ns_of(ST);
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int j = li + b * T;
            const int t0 = (j & (NS - 1)) * (N / (NS * R));
#pragma unroll
            for (int s = 1; s < R; ++s) w[b * R + s] = __ldg(tw + s * t0);
        }
    }

    // reads + twiddles + butterflies of stage ST (>= 1)
    template <int ST>
    __device__ __forceinline__ static void stage_load(const float2 *L, int li, const float2 (&w)[R0], float2 (&v)[R0])
    {
        constexpr int R = S::R[ST], B = R0 / R;
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int j = li + b * T;
            if constexpr (Map::kSwizzled && (N / R) % 64 == 0) {
                const int a = Map::at(j);
#pragma unroll
                for (int s = 0; s < R; ++s) v[b * R + s] = L[Map::shifted(a, s * (N / R))];
            } else {
#pragma unroll
                for (int s = 0; s < R; ++s) v[b * R + s] = L[Map::at(j + s * (N / R))];
            }
#pragma unroll
            for (int s = 1; s < R; ++s) v[b * R + s] = cmul(v[b * R + s], w[b * R + s]);
            Dft<R>::run(&v[b * R]);
        }
    }

    // writes of a middle stage ST (1 <= ST < NST - 1)
    template <int ST>
    __device__ __forceinline__ static void stage_store(float2 *L, int li, const float2 (&v)[R0])
    {
        constexpr int R = S::R[ST], B = R0 / R, NS = ns_of(ST);
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int j = li + b * T;
            const int o = (j / NS) * (NS * R) + (j & (NS - 1));
            if constexpr (Map::kSwizzled && NS % 64 == 0) {
                const int a = Map::at(o);
#pragma unroll
                for (int t = 0; t < R; ++t) L[Map::shifted(a, t * NS)] = v[b * R + t];
            } else {
#pragma unroll
                for (int t = 0; t < R; ++t) L[Map::at(o + t * NS)] = v[b * R + t];
            }
        }
    }

    // ---- two adjacent lines at once, kept in shared memory as float4 (line a in .xy, line b in .zw) ----
    __device__ __forceinline__ static void stage0_store2(float4 *L, int li, const float2 (&va)[R0], const float2 (&vb)[R0])
    {
#pragma unroll
        for (int t = 0; t < R0; ++t) L[Map::at(li * R0 + t)] = make_float4(va[t].x, va[t].y, vb[t].x, vb[t].y);
    }

    template <int ST>
    __device__ __forceinline__ static void stage_load2(const float4 *L, int li, const float2 (&w)[R0], float2 (&va)[R0],
                                                       float2 (&vb)[R0])
    {
        constexpr int R = S::R[ST], B = R0 / R;
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int j = li + b * T;
#pragma unroll
            for (int s = 0; s < R; ++s) {
                const float4 q = L[Map::at(j + s * (N / R))];
                va[b * R + s] = make_float2(q.x, q.y); vb[b * R + s] = make_float2(q.z, q.w);
            }
#pragma unroll
            for (int s = 1; s < R; ++s) { va[b * R + s] = cmul(va[b * R + s], w[b * R + s]); vb[b * R + s] = cmul(vb[b * R + s], w[b * R + s]); }
            Dft<R>::run(&va[b * R]);
            Dft<R>::run(&vb[b * R]);
        }
    }

    template <int ST>
    __device__ __forceinline__ static void stage_store2(float4 *L, int li, const float2 (&va)[R0], const float2 (&vb)[R0])
    {
        constexpr int R = S::R[ST], B = R0 / R, NS = ns_of(ST);
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int j = li + b * T;
            const int o = (j / NS) * (NS * R) + (j & (NS - 1));
#pragma unroll
            for (int t = 0; t < R; ++t)
                L[Map::at(o + t * NS)] = make_float4(va[b * R + t].x, va[b * R + t].y, vb[b * R + t].x, vb[b * R + t].y);
        }
    }

    // after the last stage the value of bin k = li + T m sits in v[out_reg(m)]
    __host__ __device__ static constexpr int out_reg(int m)
    {
        constexpr int R = S::R[NST - 1], B = R0 / R;
        return NST == 1 ? m : (m % B) * R + m / B;
    }
};

// Synchronises the G threads that share a line group (G a power of two; groups are aligned
// runs of thread ids).  G <= 32: the group lives inside one warp.  Otherwise a named barrier
// per group (ids 1 .. 15) unless the group is the whole CTA.
template <int G, int CTA_THREADS>
__device__ __forceinline__ void group_sync(int group)
{
    if constexpr (G <= 32) __syncwarp();
    else if constexpr (G >= CTA_THREADS) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(G) : "memory");
}

} // namespace cyr
