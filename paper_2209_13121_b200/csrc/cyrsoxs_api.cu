// cyrsoxs_api.cu -- C ABI (include/cyrsoxs.h) and host driver of the CyRSoXS hot path.
// The driver only validates, sizes buffers, computes a few per-energy scalars in double
// (k and the complex coefficients, Eq. 1 / north_star) and launches the
// kernels of kernels.cuh; every step of the path runs on the device.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <complex>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "../../include/cyrsoxs.h"
#include "kernels.cuh"
#include "kernels2.cuh"
#include "reduce.cuh"

using namespace cyr;

namespace {

constexpr double kPi = 3.141592653589793;
constexpr double kHcEvNm = 1239.84197;
constexpr int kMaxAngles = 4096;
constexpr int kMaxLog2 = 11;
constexpr int kMaxAny = 2048;           // longest axis that is not a power of two (direct DFT passes)

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
};

} // namespace

struct cyrsoxs_ctx {
    int Nx = 0, Ny = 0, Nz = 0, n_mat = 0, device = 0, n_sm = 148;
    double voxel = 0.0;
    double dqx = 0, dqy = 0, dqz = 0;
    // morphology
    MorphPtrs mp{};
    bool have_morph = false;
    std::vector<void *> owned_morph;
    // streamed mode (cyrsoxs_set_morphology_streamed): host arrays, group size, staging, events
    bool streamed = false;
    int stream_group = 0;
    MorphPtrs host_mp{};
    DevBuf stage_morph[2];
    cudaEvent_t ev_stage_ready[2] = {nullptr, nullptr}, ev_stage_free[2] = {nullptr, nullptr};
    // optics
    int nE = 0;
    std::vector<double> energies, k;
    std::vector<float> coef;           // [nE][n_mat][6]: Cc, Ca, Cb (complex) / 4 pi
    std::vector<float> reach2;         // [nE] squared reach of the valid disk in x pixels (k_rotate_avg)
    DevBuf d_coef, d_k, d_reach2;
    bool have_optics = false, optics_dirty = false;    // dirty: host tables newer than the device copies
    // angles
    int nA = 0;
    std::vector<double2> cs;
    std::vector<float4> csf;
    bool angles_dirty = false;
    DevBuf d_tiles[8];                          // rotate tile tables for EG = 1, 2, 4, 8 and AS = 1, 4
    DevBuf d_cs, d_csf;
    int n_tiles[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int eg = 1;                                 // energies interleaved per image group in this run
    unsigned long long plan_key = 0;            // what the cached energy batch was planned for
    size_t plan_fixed = 0, plan_per_e = 0;
    int plan_eb = 0;
    bool have_angles = false;
    // options
    int ewald = CYRSOXS_EWALD_TRILINEAR;
    int alg = CYRSOXS_ALG_AUTO;
    int profiling = 0;
    bool pdl = false;                  // this run launches its kernels with programmatic dependent launch (small runs)
    unsigned int *d_counts = nullptr;
    // SPECTRAL_BASIS plan (rebuilt per run from the morphology's NULL pattern and the optics)
    int n_pack = 0;
    std::vector<int> basis_kind, basis_mat;     // [2 n_pack]
    DevBuf d_bcoef, d_bkind, d_bmat;
    bool plan_dirty = true;
    // spectra shard (cyrsoxs_set_spectra_shard): this context transforms the basis fields of one contiguous group of
    // materials ("part") of n_parts; the other parts' spectra are written into the buffer by the caller (multi-GPU)
    int shard_part = 0, shard_parts = 1;
    std::vector<int> part_m0, part_m1, part_pack0, part_npack;
    int e_first = 0, e_count = -1;                  // energies processed by run / run_energies (-1: all)
    bool spectra_ready = false;                     // cyrsoxs_run_spectra has run for the current configuration
    size_t A3_pack_bytes = 0;                       // bytes of one pack's pruned spectrum in A3
    unsigned long long null_pattern = ~0ull;
    // workspace
    DevBuf A1, A2, A3, img, twx, twy, twz, stage_out[2], red;
    DevBuf tw2x;                                 // per-stage twiddle tables of fft2.cuh for the x pass (lengths 64 .. 2048)
    // last run
    cyrsoxs_stats stats{};
    cudaStream_t last_stream = nullptr;
    cudaEvent_t ev_run_done = nullptr;             // end of the last run on last_stream (cross-stream reuse of the workspace)
    bool ran = false;
    std::vector<const void *> smem_attr_done;      // kernels whose dynamic shared-memory limit has been raised
    int last_batch_e = 0;
    std::vector<cudaEvent_t> prof_events;          // pairs (start, stop) tagged by stage
    std::vector<int> prof_stage;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_batch[2] = {nullptr, nullptr}, ev_copy[2] = {nullptr, nullptr};
    std::string err;
};

namespace {

const char *kCreateFailed = "cyrsoxs_create failed (invalid argument, no CUDA device or out of memory)";

cyrsoxs_status fail(cyrsoxs_ctx *c, cyrsoxs_status st, const char *fmt, ...)
{
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    return st;
}

#define CUDA_TRY(c, expr)                                                                         \
    do {                                                                                          \
        cudaError_t _e = (expr);                                                                  \
        if (_e != cudaSuccess) {                                                                  \
            cudaGetLastError();                                                                   \
            return fail((c), _e == cudaErrorMemoryAllocation ? CYRSOXS_ERR_OOM : CYRSOXS_ERR_CUDA, \
                        "%s: %s", #expr, cudaGetErrorString(_e));                                 \
        }                                                                                         \
    } while (0)

// Makes the context's device current for the duration of an entry point and restores the caller's.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; }
        if (prev != dev) { switched = cudaSetDevice(dev) == cudaSuccess; if (!switched) cudaGetLastError(); }
    }
    ~DeviceGuard() { if (switched && prev >= 0) cudaSetDevice(prev); }
};

// Raises a kernel's dynamic shared-memory limit once per context (a context is used by one host thread).
template <class K> cyrsoxs_status allow_smem(cyrsoxs_ctx *c, K kernel, size_t bytes)
{
    const void *f = reinterpret_cast<const void *>(kernel);
    if (bytes <= 48 * 1024 || std::find(c->smem_attr_done.begin(), c->smem_attr_done.end(), f) != c->smem_attr_done.end())
        return CYRSOXS_OK;
    CUDA_TRY(c, cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    c->smem_attr_done.push_back(f);
    return CYRSOXS_OK;
}

// Launch with programmatic dependent launch allowed (sm_90+): the grid may be scheduled while the previous kernel of the
// stream is still draining; every kernel of the path starts with griddepcontrol.wait (pdl_entry() in kernels.cuh), i.e. it
// touches no memory before the previous kernel has completed and flushed -- the ordering is that of a plain stream, what
// overlaps is the launch latency and the ramp of the next grid with the tail of the last.  Measured: CFG1 31.8 -> 29.7 us,
// CFG2 109.6 -> 102.4 us per run; on large volumes the early CTAs hold SM resources idle through the long tail of the
// previous kernel (CFG3 2.74 -> 2.82 ms), so cyrsoxs_run allows it for small runs only (`pdl`).
template <class... KArgs, class... Args>
cudaError_t launch_pdl(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(std::forward<Args>(args))...);
}

bool is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }
int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

cyrsoxs_status ensure(cyrsoxs_ctx *c, DevBuf &b, size_t bytes)
{
    if (bytes <= b.cap) return CYRSOXS_OK;
    if (b.p) { cudaFree(b.p); b.p = nullptr; b.cap = 0; }
    cudaError_t e = cudaMalloc(&b.p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        b.p = nullptr;
        return fail(c, CYRSOXS_ERR_OOM, "cudaMalloc(%zu bytes): %s", bytes, cudaGetErrorString(e));
    }
    b.cap = bytes;
    return CYRSOXS_OK;
}

void release(DevBuf &b)
{
    if (b.p) cudaFree(b.p);
    b.p = nullptr; b.cap = 0;
}

// exp(-2 pi i t / N), t < N, evaluated in double and rounded once.
cyrsoxs_status make_twiddles(cyrsoxs_ctx *c, DevBuf &b, int N)
{
    std::vector<float2> h((size_t)std::max(N, 1));
    for (int t = 0; t < N; ++t) {
        double ang = -2.0 * kPi * (double)t / (double)N;
        h[t] = make_float2((float)cos(ang), (float)sin(ang));
    }
    // exact values on the axes
    if (N >= 4 && N % 4 == 0) { h[N / 4] = make_float2(0.f, -1.f); h[N / 2] = make_float2(-1.f, 0.f); h[3 * N / 4] = make_float2(0.f, 1.f); }
    else if (N % 2 == 0 && N >= 2) h[N / 2] = make_float2(-1.f, 0.f);
    cyrsoxs_status st = ensure(c, b, sizeof(float2) * h.size());
    if (st != CYRSOXS_OK) return st;
    CUDA_TRY(c, cudaMemcpy(b.p, h.data(), sizeof(float2) * h.size(), cudaMemcpyHostToDevice));
    return CYRSOXS_OK;
}

// Per-stage twiddle tables of fft2.cuh for a power-of-two length 64 .. 2048 (nothing for other lengths).
cyrsoxs_status make_twiddles2(cyrsoxs_ctx *c, DevBuf &b, int N)
{
    std::vector<float2> h;
    switch (is_pow2(N) ? ilog2(N) : 0) {
#define CASE(L) case L: h.resize(Fft2<L>::TW_TOTAL); fft2_fill_twiddles<L>(h.data()); break;
        CASE(6) CASE(7) CASE(8) CASE(9) CASE(10) CASE(11)
#undef CASE
    default: return CYRSOXS_OK;
    }
    cyrsoxs_status st = ensure(c, b, sizeof(float2) * h.size());
    if (st != CYRSOXS_OK) return st;
    CUDA_TRY(c, cudaMemcpy(b.p, h.data(), sizeof(float2) * h.size(), cudaMemcpyHostToDevice));
    return CYRSOXS_OK;
}

// Window of bins [-K, K] (symmetric) or [-K, 0] (one-sided) on an axis of length N.
Window make_window(int N, int K, bool symmetric)
{
    Window w;
    w.N = N;
    int width = symmetric ? 2 * K + 1 : K + 1;
    if (width >= N) { w.lo = -(N / 2); w.W = N; }
    else { w.lo = -K; w.W = width; }
    return w;
}

int round_up(int v, int m) { return (v + m - 1) / m * m; }

// Output tiles of the rotate kernel for image layout EG = 1 << lg and AS angle slices (slot
// lg + 4 (AS == 4)), nearest to q = 0 first (see k_rotate_avg); built on first use.
template <int AS> void rot_tile_dims(int lg, int &TW, int &TH)
{
    TW = lg == 0 ? RotMap<1, AS>::TW : lg == 1 ? RotMap<2, AS>::TW : lg == 2 ? RotMap<4, AS>::TW : RotMap<8, AS>::TW;
    TH = lg == 0 ? RotMap<1, AS>::TH : lg == 1 ? RotMap<2, AS>::TH : lg == 2 ? RotMap<4, AS>::TH : RotMap<8, AS>::TH;
}

cyrsoxs_status make_rotate_tiles(cyrsoxs_ctx *c, cudaStream_t stream, int lg, int as)
{
    const int slot = lg + (as == 4 ? 4 : 0);
    if (c->n_tiles[slot]) return CYRSOXS_OK;
    int TW, TH;
    if (as == 4) rot_tile_dims<4>(lg, TW, TH); else rot_tile_dims<1>(lg, TW, TH);
    const int ntx = (c->Nx + TW - 1) / TW, nty = (c->Ny + TH - 1) / TH;
    const double rho = (double)c->Nx / (double)c->Ny;
    std::vector<std::pair<double, uint32_t>> t;
    t.reserve((size_t)ntx * nty);
    for (int ty = 0; ty < nty; ++ty)
        for (int tx = 0; tx < ntx; ++tx) {
            const double ux = tx * TW + 0.5 * TW - c->Nx / 2, uy = (ty * TH + 0.5 * TH - c->Ny / 2) * rho;
            t.emplace_back(ux * ux + uy * uy, ((uint32_t)ty << 16) | (uint32_t)tx);
        }
    std::sort(t.begin(), t.end());
    std::vector<uint32_t> h(t.size());
    for (size_t i = 0; i < t.size(); ++i) h[i] = t[i].second;
    cyrsoxs_status st = ensure(c, c->d_tiles[slot], sizeof(uint32_t) * h.size());
    if (st != CYRSOXS_OK) return st;
    // pageable source: staged by the driver before the call returns, stream-ordered on the device
    CUDA_TRY(c, cudaMemcpyAsync(c->d_tiles[slot].p, h.data(), sizeof(uint32_t) * h.size(), cudaMemcpyHostToDevice, stream));
    c->n_tiles[slot] = (int)h.size();
    return CYRSOXS_OK;
}

// Energies interleaved per image group for a batch of eb energies: the largest of 8, 4, 2
// whose padding (lanes of the last group without an energy) stays below a third, else 1.
int choose_eg(int eb)
{
    for (int eg = 8; eg >= 2; eg >>= 1) {
        const int padded = (eb + eg - 1) / eg * eg;
        if (3 * (padded - eb) <= padded) return eg;
    }
    return 1;
}

// Windows from the largest wavenumber in [e0, e1): valid pixels have |q_x|, |q_y| <= k and
// k_z nodes in [-(k/dq_z) - 1, 0] (Eq. 8).  One extra bin of slack on every side.
void windows_for(const cyrsoxs_ctx *c, double kmax, Window &wx, Window &wy, Window &wz, int &pitch, bool sym_z = false)
{
    int Kx = (int)floor(kmax / c->dqx) + 1, Ky = (int)floor(kmax / c->dqy) + 1;
    wx = make_window(c->Nx, Kx, true);
    wy = make_window(c->Ny, Ky, true);
    if (c->Nz == 1) { wz.N = 1; wz.lo = 0; wz.W = 1; }
    else { int Kz = (int)floor(kmax / c->dqz) + 2; wz = make_window(c->Nz, Kz, sym_z); }
    pitch = round_up(wx.W, 32);
}

template <int LOGN> cyrsoxs_status launch_xpass_t(cyrsoxs_ctx *c, cudaStream_t st, int e0, int eb, float2 *out,
                                                  const Window &wx, int pitch)
{
    using Cfg = XCfg<LOGN>;
    if (cyrsoxs_status a = allow_smem(c, k_xpass_chi<LOGN>, Cfg::SMEM)) return a;
    const int rows = c->Ny * c->Nz;
    dim3 grid((rows + Cfg::ROWS - 1) / Cfg::ROWS, eb);
    launch_pdl(c->pdl, k_xpass_chi<LOGN>, grid, Cfg::THREADS, Cfg::SMEM, st, c->mp, (const float *)c->d_coef.p, e0, out, rows, wx, pitch,
                                                             (const float2 *)c->twx.p);
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

cyrsoxs_status launch_xpass(cyrsoxs_ctx *c, cudaStream_t st, int e0, int eb, float2 *out, const Window &wx, int pitch)
{
    switch (ilog2(c->Nx)) {
#define CASE(L) case L: return launch_xpass_t<L>(c, st, e0, eb, out, wx, pitch);
        CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8) CASE(9) CASE(10) CASE(11)
#undef CASE
    }
    return fail(c, CYRSOXS_ERR_INVALID_ARG, "unsupported Nx");
}

template <int LOGN> cyrsoxs_status launch_colpass_t(cyrsoxs_ctx *c, cudaStream_t st, ColParams p, int n_lo, int n_hi, int pitch)
{
    using Cfg = Col2Cfg<LOGN>;
    if (cyrsoxs_status a = allow_smem(c, k_col2<LOGN>, Cfg::SMEM)) return a;
    p.n_tiles = pitch / Cfg::TX;
    dim3 grid((unsigned)(p.n_tiles * n_lo), (unsigned)n_hi);
    launch_pdl(c->pdl, k_col2<LOGN>, grid, Cfg::THREADS, Cfg::SMEM, st, p);
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

template <int LOGN, int PW> cyrsoxs_status launch_colpass_pair_t(cyrsoxs_ctx *c, cudaStream_t st, ColParams p, int n_lo, int n_hi, int pitch)
{
    using Cfg = Col2PCfg<LOGN, PW>;
    if (cyrsoxs_status a = allow_smem(c, k_col2p<LOGN, PW>, Cfg::SMEM)) return a;
    p.n_tiles = pitch / Cfg::TX;
    dim3 grid((unsigned)(p.n_tiles * n_lo), (unsigned)n_hi);
    launch_pdl(c->pdl, k_col2p<LOGN, PW>, grid, Cfg::THREADS, Cfg::SMEM, st, p);
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

cyrsoxs_status launch_colpass(cyrsoxs_ctx *c, cudaStream_t st, int N, const ColParams &p, int n_lo, int n_hi, int pitch)
{
    if (!is_pow2(N)) {
        // an axis of any length (DESIGN 3-A14): the pruned direct DFT
        const int tx = dft_tx(N);
        const size_t smem = sizeof(float2) * ((size_t)N * tx + N);
        ColParams q = p;
        q.n_tiles = pitch / tx;
        dim3 grid((unsigned)(q.n_tiles * n_lo), (unsigned)n_hi);
        if (tx == 32) {
            if (cyrsoxs_status a = allow_smem(c, k_coldft<32>, sizeof(float2) * ((size_t)512 * 32 + 512))) return a;
            launch_pdl(c->pdl, k_coldft<32>, grid, DFT_THREADS, smem, st, q, N);
        } else {
            if (cyrsoxs_status a = allow_smem(c, k_coldft<8>, sizeof(float2) * ((size_t)kMaxAny * 8 + kMaxAny))) return a;
            launch_pdl(c->pdl, k_coldft<8>, grid, DFT_THREADS, smem, st, q, N);
        }
        CUDA_TRY(c, cudaGetLastError());
        return CYRSOXS_OK;
    }
    // lengths 128 .. 1024 take the two-columns-per-thread kernel (measured faster at every one of them:
    // cfg2 z 29 -> 25 us, cfg3 z 0.75 -> 0.65 / y 0.49 -> 0.40 ms, cfg5 z 7.4 -> 4.5 / y 4.1 -> 3.1 ms)
    constexpr int pair_min = 7;
    const int lg = ilog2(N);
#ifdef CYRSOXS_TUNING          // sweep aid, compiled out of the shipped library
    if (const char *e = getenv("CYRSOXS_PW")) {
        const int pw = atoi(e);
        if (pw == 4) switch (lg) {
            case 9: return launch_colpass_pair_t<9, 4>(c, st, p, n_lo, n_hi, pitch);
            case 10: return launch_colpass_pair_t<10, 4>(c, st, p, n_lo, n_hi, pitch);
        }
        if (pw == 2) switch (lg) {
            case 9: return launch_colpass_pair_t<9, 2>(c, st, p, n_lo, n_hi, pitch);
            case 10: return launch_colpass_pair_t<10, 2>(c, st, p, n_lo, n_hi, pitch);
        }
    }
#endif
    // all strides are multiples of 2 elements (pitch is a multiple of 32), so 128-bit accesses are aligned
    if (lg >= pair_min) {
        switch (lg) {
        case 7: return launch_colpass_pair_t<7, 8>(c, st, p, n_lo, n_hi, pitch);
        case 8: return launch_colpass_pair_t<8, 8>(c, st, p, n_lo, n_hi, pitch);
        case 9: return launch_colpass_pair_t<9, 8>(c, st, p, n_lo, n_hi, pitch);
        case 10: return launch_colpass_pair_t<10, 8>(c, st, p, n_lo, n_hi, pitch);
        }
    }
    switch (lg) {
#define CASE(L) case L: return launch_colpass_t<L>(c, st, p, n_lo, n_hi, pitch);
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8) CASE(9) CASE(10) CASE(11)
#undef CASE
    }
    return fail(c, CYRSOXS_ERR_INVALID_ARG, "unsupported transform length %d", N);
}

struct StageTimer {
    cyrsoxs_ctx *c;
    cudaStream_t st;
    int stage;
    cudaEvent_t a = nullptr, b = nullptr;
    StageTimer(cyrsoxs_ctx *c_, cudaStream_t s, int stage_) : c(c_), st(s), stage(stage_)
    {
        c->stats.stage_launches[stage]++;
        c->stats.kernel_launches++;
        if (c->profiling) {
            cudaEventCreate(&a); cudaEventCreate(&b);
            cudaEventRecord(a, st);
        }
    }
    ~StageTimer()
    {
        if (c->profiling) {
            cudaEventRecord(b, st);
            c->prof_events.push_back(a); c->prof_events.push_back(b);
            c->prof_stage.push_back(stage);
        }
    }
};

void clear_prof(cyrsoxs_ctx *c)
{
    for (cudaEvent_t e : c->prof_events) cudaEventDestroy(e);
    c->prof_events.clear();
    c->prof_stage.clear();
}

template <int EG> dim3 ewald_grid(const cyrsoxs_ctx *c, int eb)
{
    using M = EwaldMap<EG>;
    return dim3((c->Nx + M::PW - 1) / M::PW, (c->Ny + M::PH - 1) / M::PH, (eb + EG - 1) / EG);
}

template <int EG>
cyrsoxs_status launch_rotate_t(cyrsoxs_ctx *c, cudaStream_t st, RotateParams p, int eb, int lg)
{
    // groups per CTA: all of them (up to ROT_GMAX), so the cells of an angle are computed once per pixel
    const int ng = (eb + EG - 1) / EG;
    const int gpc = std::min(ng, ROT_GMAX);
    const int slices_y = (ng + gpc - 1) / gpc;
    p.gpc = gpc;
    // angle slices: 4 threads per pixel when one per pixel leaves the machine under-filled and there are
    // several energy groups to walk through per angle (cfg2: 38 -> 35 us; no gain on cfg1's single energy)
    const long long px_ctas = ((long long)c->Nx * c->Ny * EG + 255) / 256 * slices_y;
    int as = (px_ctas < 4LL * c->n_sm && c->nA >= 8 && ng >= 2) ? 4 : 1;
    cyrsoxs_status s = make_rotate_tiles(c, st, lg, as);
    if (s != CYRSOXS_OK) return s;
    const int slot = lg + (as == 4 ? 4 : 0);
    p.tiles = (const uint32_t *)c->d_tiles[slot].p;
    const dim3 grid((unsigned)c->n_tiles[slot], slices_y);
    const size_t smem = (size_t)gpc * 256 * 8;
    // angles in flight: 1 when the grid fills the machine several times over (occupancy hides the
    // load latency; measured best on cfg4), more when it does not
    const int ua = (long long)grid.x * grid.y >= 16LL * c->n_sm ? 1 : (as == 4 ? 2 : 4);
    if (as == 4) {
        if (ua == 4) launch_pdl(c->pdl, k_rotate_avg<EG, 4, 2, 4>, grid, 256, smem, st, p);
        else if (ua == 2) launch_pdl(c->pdl, k_rotate_avg<EG, 2, 3, 4>, grid, 256, smem, st, p);
        else launch_pdl(c->pdl, k_rotate_avg<EG, 1, 4, 4>, grid, 256, smem, st, p);
    } else {
        if (ua == 4) launch_pdl(c->pdl, k_rotate_avg<EG, 4, 2, 1>, grid, 256, smem, st, p);
        else if (ua == 2) launch_pdl(c->pdl, k_rotate_avg<EG, 2, 3, 1>, grid, 256, smem, st, p);
        else launch_pdl(c->pdl, k_rotate_avg<EG, 1, 4, 1>, grid, 256, smem, st, p);
    }
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

// Rotate back + average for energies [e0, e0 + eb) of the image buffer.
cyrsoxs_status launch_rotate(cyrsoxs_ctx *c, cudaStream_t st, int e0, int eb, float *d_out, unsigned int *d_cnt)
{
    StageTimer t(c, st, CYRSOXS_STAGE_ROTATE);
    RotateParams p{};
    p.Nx = c->Nx; p.Ny = c->Ny; p.n_angles = c->nA; p.n_energy = eb;
    p.cs = (const double2 *)c->d_cs.p; p.csf = (const float4 *)c->d_csf.p;
    p.img = (const float4 *)c->img.p; p.out = d_out; p.counts = d_cnt;
    p.reach2 = (const float *)c->d_reach2.p + e0;
    p.rho = (double)c->Nx / (double)c->Ny;
    cyrsoxs_status s;
    switch (c->eg) {
    case 8: s = launch_rotate_t<8>(c, st, p, eb, 3); break;
    case 4: s = launch_rotate_t<4>(c, st, p, eb, 2); break;
    case 2: s = launch_rotate_t<2>(c, st, p, eb, 1); break;
    default: s = launch_rotate_t<1>(c, st, p, eb, 0); break;
    }
    if (s != CYRSOXS_OK) return s;
    c->stats.stage_bytes[CYRSOXS_STAGE_ROTATE] += eb * (20.0 * c->Nx * c->Ny);
    return CYRSOXS_OK;
}

// One energy batch of the PER_ENERGY algorithm: fields -> x -> z -> y -> Ewald -> rotate.
cyrsoxs_status run_batch_per_energy(cyrsoxs_ctx *c, cudaStream_t st, int e0, int eb, float *d_out, unsigned int *d_cnt)
{
    double kmax = 0;
    for (int e = e0; e < e0 + eb; ++e) kmax = std::max(kmax, c->k[e]);
    Window wx, wy, wz;
    int pitch;
    windows_for(c, kmax, wx, wy, wz, pitch);
    const int F = NCHI * eb;
    const size_t rows = (size_t)c->Ny * c->Nz;
    float2 *A1 = (float2 *)c->A1.p, *A2 = (float2 *)c->A2.p, *A3 = (float2 *)c->A3.p;
    cyrsoxs_status s;
    double n_iso = 0, n_al = 0;
    for (int m = 0; m < c->n_mat; ++m) (c->mp.S[m] ? n_al : n_iso) += 1;
    const double nvox = (double)c->Nx * c->Ny * c->Nz;
    {
        StageTimer t(c, st, CYRSOXS_STAGE_XPASS);
        if ((s = launch_xpass(c, st, e0, eb, A1, wx, pitch)) != CYRSOXS_OK) return s;
        c->stats.stage_bytes[CYRSOXS_STAGE_XPASS] += eb * nvox * (16.0 * n_al + 4.0 * n_iso) + 8.0 * F * rows * pitch;
    }
    const float2 *ysrc = A1;
    if (c->Nz > 1) {
        StageTimer t(c, st, CYRSOXS_STAGE_ZPASS);
        ColParams p{};
        p.in = A1; p.out = A2;
        p.in_row = (long long)c->Ny * pitch; p.out_row = (long long)c->Ny * pitch;
        p.in_lo = pitch; p.out_lo = pitch;
        p.in_hi = (long long)c->Nz * c->Ny * pitch; p.out_hi = (long long)wz.W * c->Ny * pitch;
        p.win = wz; p.tw = (const float2 *)c->twz.p;
        if ((s = launch_colpass(c, st, c->Nz, p, c->Ny, F, pitch)) != CYRSOXS_OK) return s;
        c->stats.stage_bytes[CYRSOXS_STAGE_ZPASS] += 8.0 * F * c->Ny * pitch * ((double)c->Nz + wz.W);
        ysrc = A2;
    }
    {
        StageTimer t(c, st, CYRSOXS_STAGE_YPASS);
        ColParams p{};
        p.in = ysrc; p.out = A3;
        p.in_row = pitch; p.out_row = pitch;
        p.in_lo = (long long)c->Ny * pitch; p.out_lo = (long long)wy.W * pitch;
        p.in_hi = (long long)wz.W * c->Ny * pitch; p.out_hi = (long long)wz.W * wy.W * pitch;
        p.win = wy; p.tw = (const float2 *)c->twy.p;
        if ((s = launch_colpass(c, st, c->Ny, p, wz.W, F, pitch)) != CYRSOXS_OK) return s;
        c->stats.stage_bytes[CYRSOXS_STAGE_YPASS] += 8.0 * F * wz.W * pitch * ((double)c->Ny + wy.W);
    }
    {
        StageTimer t(c, st, CYRSOXS_STAGE_EWALD);
        EwaldParams p{};
        p.Nx = c->Nx; p.Ny = c->Ny; p.Nz = c->Nz; p.mode = c->ewald;
        p.dqx = c->dqx; p.dqy = c->dqy; p.dqz = c->dqz;
        p.k = (const double *)c->d_k.p; p.e0 = e0; p.n_e = eb;
        p.wx = wx; p.wy = wy; p.wz = wz; p.pitch = pitch;
        p.spec = A3; p.img = (float4 *)c->img.p;
        switch (c->eg) {
#define CASE(EG) case EG: launch_pdl(c->pdl, k_ewald_chi<EG>, ewald_grid<EG>(c, eb), 256, 0, st, p); break;
            CASE(8) CASE(4) CASE(2) default: CASE(1)
#undef CASE
        }
        CUDA_TRY(c, cudaGetLastError());
        const double nodes = (c->Nz > 1 && c->ewald == CYRSOXS_EWALD_TRILINEAR) ? 2.0 : 1.0;
        c->stats.stage_bytes[CYRSOXS_STAGE_EWALD] += eb * ((double)wx.W * wy.W * (kPi / 4.0) * nodes * NCHI * 8.0 + 16.0 * c->Nx * c->Ny);
    }
    return launch_rotate(c, st, e0, eb, d_out, d_cnt);
}

// rows: rows (of Nx voxels) this launch transforms, starting at the morphology pointers of `mp`; fstride: distance
// (float2 elements) between the packs of `out`.
template <int LOGN> cyrsoxs_status launch_xbasis_t(cyrsoxs_ctx *c, cudaStream_t st, const MorphPtrs &mp, float2 *out, const Window &wx, int pitch,
                                                   int rows, size_t fstride)
{
    using Cfg = XB2Cfg<LOGN>;
    if (cyrsoxs_status a = allow_smem(c, k_xbasis2<LOGN>, Cfg::SMEM)) return a;
    dim3 grid((rows + Cfg::ROWS - 1) / Cfg::ROWS);
    launch_pdl(c->pdl, k_xbasis2<LOGN>, grid, Cfg::THREADS, Cfg::SMEM, st, mp, out, rows, fstride, wx, pitch, (const float2 *)c->twx.p);
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

template <int LOGN> cyrsoxs_status launch_xbasis3_t(cyrsoxs_ctx *c, cudaStream_t st, const MorphPtrs &mp, float2 *out, const Window &wx, int pitch,
                                                    int rows, size_t fstride)
{
    using Cfg = XB3Cfg<LOGN>;
    if (cyrsoxs_status a = allow_smem(c, k_xbasis3<LOGN>, Cfg::SMEM)) return a;
    dim3 grid((rows + Cfg::ROWS - 1) / Cfg::ROWS);
    size_t smem = Cfg::SMEM;
#ifdef CYRSOXS_TUNING          // sweep aid, compiled out of the shipped library: occupancy sensitivity
    if (const char *e = getenv("CYRSOXS_XB3_SMEM")) { smem = std::max(smem, (size_t)atoi(e)); cudaFuncSetAttribute(k_xbasis3<LOGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024); }
#endif
    int ahead = c->n_sm * Cfg::MINB * Cfg::ROWS;               // rows in flight on the whole GPU
#ifdef CYRSOXS_TUNING
    if (const char *e = getenv("CYRSOXS_XB3_AHEAD")) ahead = atoi(e);
#endif
    launch_pdl(c->pdl, k_xbasis3<LOGN>, grid, Cfg::THREADS, smem, st, mp, out, rows, fstride, wx, pitch, (const float2 *)c->tw2x.p, ahead);
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

// pack0 / mat0: first pack and first material of `mp` in the basis plan (non-zero for the material groups of the streamed mode)
cyrsoxs_status launch_xbasis(cyrsoxs_ctx *c, cudaStream_t st, const MorphPtrs &mp, float2 *out, const Window &wx, int pitch,
                             int rows, size_t fstride, int pack0 = 0, int mat0 = 0, int n_pack = -1)
{
    if (!is_pow2(c->Nx)) {
        // a row length that is not a power of two: direct DFT at the window's bins (k_xdft)
        const size_t smem = sizeof(float2) * 2 * (size_t)c->Nx;
        if (n_pack < 0) n_pack = c->n_pack;
        launch_pdl(c->pdl, k_xdft, rows, XDFT_THREADS, smem, st, mp, (const int *)c->d_bkind.p + 2 * pack0, (const int *)c->d_bmat.p + 2 * pack0, mat0, n_pack, out,
                                                 rows, fstride, wx, pitch, (const float2 *)c->twx.p, c->Nx);
        CUDA_TRY(c, cudaGetLastError());
        return CYRSOXS_OK;
    }
    switch (ilog2(c->Nx)) {
#define CASE3(L) case L: return launch_xbasis3_t<L>(c, st, mp, out, wx, pitch, rows, fstride);
        CASE3(6) CASE3(7) CASE3(8) CASE3(9) CASE3(10) CASE3(11)
#undef CASE3
#define CASE(L) case L: return launch_xbasis_t<L>(c, st, mp, out, wx, pitch, rows, fstride);
        CASE(2) CASE(3) CASE(4) CASE(5)
#undef CASE
    }
    return fail(c, CYRSOXS_ERR_INVALID_ARG, "unsupported Nx");
}

// Device copies of the small host tables (per-energy coefficients and wavenumbers, per-angle cos/sin) are refreshed
// at cyrsoxs_run, on the run's stream: a setter called while an earlier run is still executing cannot overwrite what
// that run's kernels read (the copies are ordered after it on the stream).  Pageable sources are staged by the
// driver before cudaMemcpyAsync returns, so the host vectors may change right afterwards.
cyrsoxs_status upload_tables(cyrsoxs_ctx *c, cudaStream_t st)
{
    cyrsoxs_status s;
    if (c->optics_dirty) {
        if ((s = ensure(c, c->d_coef, sizeof(float) * c->coef.size())) != CYRSOXS_OK) return s;
        if ((s = ensure(c, c->d_k, sizeof(double) * c->k.size())) != CYRSOXS_OK) return s;
        if ((s = ensure(c, c->d_reach2, sizeof(float) * c->reach2.size())) != CYRSOXS_OK) return s;
        CUDA_TRY(c, cudaMemcpyAsync(c->d_coef.p, c->coef.data(), sizeof(float) * c->coef.size(), cudaMemcpyHostToDevice, st));
        CUDA_TRY(c, cudaMemcpyAsync(c->d_k.p, c->k.data(), sizeof(double) * c->k.size(), cudaMemcpyHostToDevice, st));
        CUDA_TRY(c, cudaMemcpyAsync(c->d_reach2.p, c->reach2.data(), sizeof(float) * c->reach2.size(), cudaMemcpyHostToDevice, st));
        c->optics_dirty = false;
    }
    if (c->angles_dirty) {
        if ((s = ensure(c, c->d_cs, sizeof(double2) * c->cs.size())) != CYRSOXS_OK) return s;
        if ((s = ensure(c, c->d_csf, sizeof(float4) * c->csf.size())) != CYRSOXS_OK) return s;
        CUDA_TRY(c, cudaMemcpyAsync(c->d_cs.p, c->cs.data(), sizeof(double2) * c->cs.size(), cudaMemcpyHostToDevice, st));
        CUDA_TRY(c, cudaMemcpyAsync(c->d_csf.p, c->csf.data(), sizeof(float4) * c->csf.size(), cudaMemcpyHostToDevice, st));
        c->angles_dirty = false;
    }
    return CYRSOXS_OK;
}

// Is material m aligned (has S, theta, psi)?  In streamed mode the host table decides.
bool is_aligned(const cyrsoxs_ctx *c, int m) { return (c->streamed ? c->host_mp.S[m] : c->mp.S[m]) != nullptr; }

// The basis fields in material order (7 per aligned, 1 per isotropic material), two per complex
// pack, the last pack padded; the per-field kind/material tables and the per-energy complex
// coefficient of each field (times 1/2 for the unpacking).
cyrsoxs_status build_basis_plan(cyrsoxs_ctx *c, cudaStream_t st)
{
    c->basis_kind.clear(); c->basis_mat.clear();
    // parts of a spectra shard: contiguous material ranges of about equal field count (7 per aligned, 1 per isotropic
    // material), every part at least one material
    const int P = c->streamed ? 1 : c->shard_parts;
    c->part_m0.assign(P, 0); c->part_m1.assign(P, 0); c->part_pack0.assign(P, 0); c->part_npack.assign(P, 0);
    {
        int total = 0;
        for (int m = 0; m < c->n_mat; ++m) total += is_aligned(c, m) ? 7 : 1;
        int m = 0, cum = 0;
        for (int q = 0; q < P; ++q) {
            c->part_m0[q] = m;
            const int must_leave = P - 1 - q;                 // materials the later parts need
            const long long target = (long long)total * (q + 1);      // cumulative field count the part should end at, times P
            for (;;) {
                cum += is_aligned(c, m) ? 7 : 1; ++m;
                if (m >= c->n_mat - must_leave) break;
                // take the next material too if that ends closer to the target (the last part takes everything left)
                const long long next = (long long)(cum + (is_aligned(c, m) ? 7 : 1)) * P - target, now = (long long)cum * P - target;
                if (q < P - 1 && llabs(next) >= llabs(now)) break;
            }
            c->part_m1[q] = m;
        }
    }
    int part = 0;
    for (int m = 0; m < c->n_mat; ++m) {
        if (P > 1 && m == c->part_m0[part]) c->part_pack0[part] = (int)c->basis_kind.size() / 2;
        if (is_aligned(c, m)) for (int kd = BK_PHI; kd <= BK_YZ; ++kd) { c->basis_kind.push_back(kd); c->basis_mat.push_back(m); }
        else { c->basis_kind.push_back(BK_PHI); c->basis_mat.push_back(m); }
        // streamed mode / sharded spectra: every material group is transformed by its own launch (on its own GPU), so its
        // fields are paired among themselves and an odd count is padded at the group's end
        const bool group_end = (c->streamed && ((m + 1) % c->stream_group == 0)) || (P > 1 && m + 1 == c->part_m1[part]);
        if (group_end && (c->basis_kind.size() & 1)) { c->basis_kind.push_back(BK_NONE); c->basis_mat.push_back(0); }
        if (P > 1 && m + 1 == c->part_m1[part]) { c->part_npack[part] = (int)c->basis_kind.size() / 2 - c->part_pack0[part]; ++part; }
    }
    if (c->basis_kind.size() & 1) { c->basis_kind.push_back(BK_NONE); c->basis_mat.push_back(0); }
    const int pack = (int)c->basis_kind.size() / 2;
    c->n_pack = pack;
    if (P == 1) { c->part_m1[0] = c->n_mat; c->part_npack[0] = pack; }
    c->spectra_ready = false;
    const int nb = 2 * pack;
    std::vector<float2> coef((size_t)c->nE * nb);
    for (int e = 0; e < c->nE; ++e)
        for (int b = 0; b < nb; ++b) {
            const float *o = &c->coef[((size_t)e * c->n_mat + c->basis_mat[b]) * 6];
            float2 v = make_float2(0.f, 0.f);
            switch (c->basis_kind[b]) {
            case BK_PHI: v = make_float2(o[0], o[1]); break;
            case BK_W: v = make_float2(o[2], o[3]); break;
            case BK_NONE: break;
            default: v = make_float2(o[4], o[5]); break;
            }
            coef[(size_t)e * nb + b] = make_float2(0.5f * v.x, 0.5f * v.y);
        }
    cyrsoxs_status s;
    if ((s = ensure(c, c->d_bcoef, sizeof(float2) * coef.size())) != CYRSOXS_OK) return s;
    if ((s = ensure(c, c->d_bkind, sizeof(int) * nb)) != CYRSOXS_OK) return s;
    if ((s = ensure(c, c->d_bmat, sizeof(int) * nb)) != CYRSOXS_OK) return s;
    // pageable sources: staged by the driver before these calls return; ordered after the stream's earlier work
    CUDA_TRY(c, cudaMemcpyAsync(c->d_bcoef.p, coef.data(), sizeof(float2) * coef.size(), cudaMemcpyHostToDevice, st));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_bkind.p, c->basis_kind.data(), sizeof(int) * nb, cudaMemcpyHostToDevice, st));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_bmat.p, c->basis_mat.data(), sizeof(int) * nb, cudaMemcpyHostToDevice, st));
    c->plan_dirty = false;
    return CYRSOXS_OK;
}

// Spectra of all basis packs: x -> z -> y, once per run.  A3 = [pack][wz][wy][pitch].
cyrsoxs_status run_basis_spectra(cyrsoxs_ctx *c, cudaStream_t st, const Window &wx, const Window &wy, const Window &wz, int pitch)
{
    const size_t rows = (size_t)c->Ny * c->Nz;
    // this context's part of the basis (all of it unless a spectra shard is set): packs [pk0, pk0 + F), materials [m0, m1)
    const bool sharded = !c->streamed && c->shard_parts > 1;
    const int pk0 = sharded ? c->part_pack0[c->shard_part] : 0, F = sharded ? c->part_npack[c->shard_part] : c->n_pack;
    const int m0s = sharded ? c->part_m0[c->shard_part] : 0, m1s = sharded ? c->part_m1[c->shard_part] : c->n_mat;
    const size_t fstride1 = rows * (size_t)pitch;
    float2 *A1 = (float2 *)c->A1.p + (size_t)pk0 * fstride1;
    float2 *A2 = (float2 *)c->A2.p + (c->Nz > 1 ? (size_t)pk0 * wz.W * c->Ny * pitch : 0);
    float2 *A3 = (float2 *)c->A3.p + (size_t)pk0 * wz.W * wy.W * pitch;
    const double nvox = (double)c->Nx * c->Ny * c->Nz;
    cyrsoxs_status s;
    double n_iso = 0, n_al = 0;
    for (int m = m0s; m < m1s; ++m) (is_aligned(c, m) ? n_al : n_iso) += 1;
    if (!c->streamed) {
        StageTimer t(c, st, CYRSOXS_STAGE_XPASS);
        MorphPtrs sub = c->mp;
        if (sharded) {
            sub = MorphPtrs{};
            sub.n_mat = m1s - m0s;
            for (int m = m0s; m < m1s; ++m) {
                sub.phi[m - m0s] = c->mp.phi[m]; sub.S[m - m0s] = c->mp.S[m]; sub.theta[m - m0s] = c->mp.theta[m]; sub.psi[m - m0s] = c->mp.psi[m];
            }
        }
        if ((s = launch_xbasis(c, st, sub, A1, wx, pitch, (int)rows, fstride1, pk0, m0s, F)) != CYRSOXS_OK) return s;
    } else {
        // Memory-minimising mode (the paper's Algorithm 2/3 idea): material groups are
        // uploaded into a double-buffered staging area on the copy stream while the previous group's
        // fields are transformed on `st`; the spectra play the role of N_t.
        const size_t nv = (size_t)c->Nx * c->Ny * c->Nz, abytes = sizeof(float) * nv;
        const int G = c->stream_group;
        if (!c->copy_stream) CUDA_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            if ((s = ensure(c, c->stage_morph[i], abytes * 4 * (size_t)G)) != CYRSOXS_OK) return s;
            if (!c->ev_stage_ready[i]) CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_stage_ready[i], cudaEventDisableTiming));
            if (!c->ev_stage_free[i]) CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_stage_free[i], cudaEventDisableTiming));
        }
        const size_t fstride = fstride1;
        int pack0 = 0, g = 0;
        for (int m0 = 0; m0 < c->n_mat; m0 += G, ++g) {
            const int slot = g & 1, m1 = std::min(c->n_mat, m0 + G);
            // the slot is free once the x pass that last read it (two groups ago, or in the previous run) is done
            CUDA_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->ev_stage_free[slot], 0));
            MorphPtrs sub{};
            sub.n_mat = m1 - m0;
            float *base = (float *)c->stage_morph[slot].p;
            int fields = 0;
            for (int m = m0; m < m1; ++m) {
                const float *src[4] = {c->host_mp.phi[m], c->host_mp.S[m], c->host_mp.theta[m], c->host_mp.psi[m]};
                const float *dst[4] = {nullptr, nullptr, nullptr, nullptr};
                for (int j = 0; j < 4; ++j) {
                    if (!src[j]) continue;
                    float *d = base + ((size_t)(m - m0) * 4 + j) * nv;
                    CUDA_TRY(c, cudaMemcpyAsync(d, src[j], abytes, cudaMemcpyHostToDevice, c->copy_stream));
                    dst[j] = d;
                }
                sub.phi[m - m0] = dst[0]; sub.S[m - m0] = dst[1]; sub.theta[m - m0] = dst[2]; sub.psi[m - m0] = dst[3];
                fields += src[1] ? 7 : 1;
            }
            CUDA_TRY(c, cudaEventRecord(c->ev_stage_ready[slot], c->copy_stream));
            CUDA_TRY(c, cudaStreamWaitEvent(st, c->ev_stage_ready[slot], 0));
            {
                StageTimer t(c, st, CYRSOXS_STAGE_XPASS);
                if ((s = launch_xbasis(c, st, sub, A1 + (size_t)pack0 * fstride, wx, pitch, (int)rows, fstride, pack0, m0, (fields + 1) / 2)) != CYRSOXS_OK) return s;
            }
            CUDA_TRY(c, cudaEventRecord(c->ev_stage_free[slot], st));
            pack0 += (fields + 1) / 2;
        }
    }
    c->stats.stage_bytes[CYRSOXS_STAGE_XPASS] += nvox * (16.0 * n_al + 4.0 * n_iso) + 8.0 * F * rows * pitch;
    const float2 *ysrc = A1;
    if (c->Nz > 1) {
        StageTimer t(c, st, CYRSOXS_STAGE_ZPASS);
        ColParams p{};
        p.in = A1; p.out = A2;
        p.in_row = (long long)c->Ny * pitch; p.out_row = (long long)c->Ny * pitch;
        p.in_lo = pitch; p.out_lo = pitch;
        p.in_hi = (long long)c->Nz * c->Ny * pitch; p.out_hi = (long long)wz.W * c->Ny * pitch;
        p.win = wz; p.tw = (const float2 *)c->twz.p;
        if ((s = launch_colpass(c, st, c->Nz, p, c->Ny, F, pitch)) != CYRSOXS_OK) return s;
        c->stats.stage_bytes[CYRSOXS_STAGE_ZPASS] += 8.0 * F * c->Ny * pitch * ((double)c->Nz + wz.W);
        ysrc = A2;
    }
    {
        StageTimer t(c, st, CYRSOXS_STAGE_YPASS);
        ColParams p{};
        p.in = ysrc; p.out = A3;
        p.in_row = pitch; p.out_row = pitch;
        p.in_lo = (long long)c->Ny * pitch; p.out_lo = (long long)wy.W * pitch;
        p.in_hi = (long long)wz.W * c->Ny * pitch; p.out_hi = (long long)wz.W * wy.W * pitch;
        p.win = wy; p.tw = (const float2 *)c->twy.p;
        if ((s = launch_colpass(c, st, c->Ny, p, wz.W, F, pitch)) != CYRSOXS_OK) return s;
        c->stats.stage_bytes[CYRSOXS_STAGE_YPASS] += 8.0 * F * wz.W * pitch * ((double)c->Ny + wy.W);
    }
    return CYRSOXS_OK;
}

// One energy batch of SPECTRAL_BASIS: shell gather + rotate.
cyrsoxs_status run_batch_spectral(cyrsoxs_ctx *c, cudaStream_t st, int e0, int eb, const Window &wx, const Window &wy,
                                  const Window &wz, int pitch, float *d_out, unsigned int *d_cnt)
{
    {
        StageTimer t(c, st, CYRSOXS_STAGE_EWALD);
        EwaldBasisParams q{};
        EwaldParams &p = q.g;
        p.Nx = c->Nx; p.Ny = c->Ny; p.Nz = c->Nz; p.mode = c->ewald;
        p.dqx = c->dqx; p.dqy = c->dqy; p.dqz = c->dqz;
        p.k = (const double *)c->d_k.p; p.e0 = e0; p.n_e = eb;
        p.wx = wx; p.wy = wy; p.wz = wz; p.pitch = pitch;
        p.spec = (const float2 *)c->A3.p; p.img = (float4 *)c->img.p;
        q.n_pack = c->n_pack; q.coef = (const float2 *)c->d_bcoef.p; q.kind = (const int *)c->d_bkind.p;
        const size_t smem2d = (size_t)eb * (2 * sizeof(double) + sizeof(float) + 2 * c->n_pack * sizeof(float2)) + 2 * c->n_pack * sizeof(int)
                              + (size_t)2 * c->n_pack * 256 * sizeof(float2);
        const bool two_d = c->Nz == 1 && eb >= 4 && 2 * c->n_pack <= EW2D_MAXF && smem2d <= 96 * 1024;
        if (two_d) {
            // 2-D model, several energies: one thread per pixel, the batch's energies in an inner loop (see
            // k_ewald_basis_2d; cfg4 15.8 -> 6.6 ms; a single energy is better off with a thread per energy)
            const dim3 g2d((c->Nx + 31) / 32, (c->Ny + 7) / 8);
            switch (c->eg) {
#define CASE(EG) case EG: if (cyrsoxs_status a = allow_smem(c, k_ewald_basis_2d<EG>, 96 * 1024)) return a; launch_pdl(c->pdl, k_ewald_basis_2d<EG>, g2d, 256, smem2d, st, q); break;
                CASE(8) CASE(4) CASE(2) default: CASE(1)
#undef CASE
            }
        } else {
            switch (c->eg) {
#define CASE(EG) case EG: launch_pdl(c->pdl, k_ewald_basis<EG>, ewald_grid<EG>(c, eb), 256, 0, st, q); break;
                CASE(8) CASE(4) CASE(2) default: CASE(1)
#undef CASE
            }
        }
        CUDA_TRY(c, cudaGetLastError());
        const double nodes = (c->Nz > 1 && c->ewald == CYRSOXS_EWALD_TRILINEAR) ? 2.0 : 1.0;
        // gather: the valid disk's share (pi/4) of the spectral window, both partner bins of every pack; the 2-D kernel
        // gathers once per BATCH (its energies loop over the unpacked fields in shared memory), the 3-D one per energy.
        // Plus one float4 image per pixel and energy.
        const double gather = (double)wx.W * wy.W * (kPi / 4.0) * nodes * 2.0 * c->n_pack * 8.0;
        c->stats.stage_bytes[CYRSOXS_STAGE_EWALD] += (two_d ? 1.0 : (double)eb) * gather + (double)eb * 16.0 * c->Nx * c->Ny;
    }
    return launch_rotate(c, st, e0, eb, d_out, d_cnt);
}

} // namespace

// =========================================================================================

extern "C" {

const char *cyrsoxs_version(void) { return "cyrsoxs-b200 0.1 (sm_100a)"; }

const char *cyrsoxs_last_error(const cyrsoxs_ctx *ctx) { return ctx ? ctx->err.c_str() : kCreateFailed; }

cyrsoxs_status cyrsoxs_create(int Nx, int Ny, int Nz, int n_mat, double voxel_nm, cyrsoxs_ctx **out)
{
    if (!out) return CYRSOXS_ERR_INVALID_ARG;
    *out = nullptr;
    const int maxn = 1 << kMaxLog2;
    static_assert(kMaxAny <= (1 << kMaxLog2), "direct-DFT passes cover every accepted length");
    if (Nx < 4 || Ny < 2 || Nz < 1 || Nx > maxn || Ny > maxn || Nz > maxn) return CYRSOXS_ERR_INVALID_ARG;      // DESIGN 3-A14
    if (n_mat < 1 || n_mat > MAX_MAT || !(voxel_nm > 0.0) || !isfinite(voxel_nm)) return CYRSOXS_ERR_INVALID_ARG;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return CYRSOXS_ERR_CUDA; }
    cyrsoxs_ctx *c = new (std::nothrow) cyrsoxs_ctx();
    if (!c) return CYRSOXS_ERR_OOM;
    c->Nx = Nx; c->Ny = Ny; c->Nz = Nz; c->n_mat = n_mat; c->voxel = voxel_nm; c->device = dev;
    c->dqx = (2.0 * kPi) / ((double)Nx * voxel_nm);
    c->dqy = (2.0 * kPi) / ((double)Ny * voxel_nm);
    c->dqz = (2.0 * kPi) / ((double)Nz * voxel_nm);
    c->mp.n_mat = n_mat;
    if (cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); c->n_sm = 148; }
    cyrsoxs_status st;
    if ((st = make_twiddles(c, c->twx, Nx)) != CYRSOXS_OK || (st = make_twiddles(c, c->twy, Ny)) != CYRSOXS_OK
        || (st = make_twiddles(c, c->twz, Nz)) != CYRSOXS_OK || (st = make_twiddles2(c, c->tw2x, Nx)) != CYRSOXS_OK) {
        cyrsoxs_destroy(c);
        return st;
    }
    *out = c;
    return CYRSOXS_OK;
}

void cyrsoxs_destroy(cyrsoxs_ctx *c)
{
    if (!c) return;
    DeviceGuard guard(c->device);
    cudaDeviceSynchronize();                 // nothing of this context may still be running when its buffers go
    clear_prof(c);
    for (void *p : c->owned_morph) cudaFree(p);
    for (DevBuf *b : {&c->d_coef, &c->d_k, &c->d_reach2, &c->d_cs, &c->d_csf, &c->d_tiles[0], &c->d_tiles[1], &c->d_tiles[2], &c->d_tiles[3], &c->d_tiles[4], &c->d_tiles[5], &c->d_tiles[6], &c->d_tiles[7], &c->A1, &c->A2, &c->A3, &c->img, &c->twx, &c->twy, &c->twz, &c->tw2x,
                      &c->stage_out[0], &c->stage_out[1], &c->d_bcoef, &c->d_bkind, &c->d_bmat, &c->red})
        release(*b);
    release(c->stage_morph[0]); release(c->stage_morph[1]);
    for (int i = 0; i < 2; ++i) {
        if (c->ev_stage_ready[i]) cudaEventDestroy(c->ev_stage_ready[i]);
        if (c->ev_stage_free[i]) cudaEventDestroy(c->ev_stage_free[i]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->ev_run_done) cudaEventDestroy(c->ev_run_done);
    for (int i = 0; i < 2; ++i) {
        if (c->ev_batch[i]) cudaEventDestroy(c->ev_batch[i]);
        if (c->ev_copy[i]) cudaEventDestroy(c->ev_copy[i]);
    }
    delete c;
}

static void note_null_pattern(cyrsoxs_ctx *c)
{
    c->spectra_ready = false;                // called by every morphology setter: the spectra belong to the old morphology
    unsigned long long pat = 0;
    for (int m = 0; m < c->n_mat; ++m) pat |= (unsigned long long)is_aligned(c, m) << m;
    if (c->streamed) pat ^= 0x8000000000000000ull ^ ((unsigned long long)c->stream_group << 40);
    if (pat != c->null_pattern) { c->null_pattern = pat; c->plan_dirty = true; }
}

static cyrsoxs_status check_morph_tables(cyrsoxs_ctx *c, const float *const *phi, const float *const *S,
                                         const float *const *theta, const float *const *psi)
{
    if (!phi) return fail(c, CYRSOXS_ERR_INVALID_ARG, "phi table is NULL");
    for (int m = 0; m < c->n_mat; ++m) {
        if (!phi[m]) return fail(c, CYRSOXS_ERR_INVALID_ARG, "phi[%d] is NULL", m);
        const float *s = S ? S[m] : nullptr, *t = theta ? theta[m] : nullptr, *p = psi ? psi[m] : nullptr;
        if ((s || t || p) && !(s && t && p))
            return fail(c, CYRSOXS_ERR_INVALID_ARG, "material %d: S, theta, psi must be all set or all NULL", m);
    }
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_morphology(cyrsoxs_ctx *c, const float *const *d_phi, const float *const *d_S,
                                      const float *const *d_theta, const float *const *d_psi)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    cyrsoxs_status st = check_morph_tables(c, d_phi, d_S, d_theta, d_psi);
    if (st != CYRSOXS_OK) return st;
    for (int m = 0; m < c->n_mat; ++m) {
        const float *ptrs[4] = {d_phi[m], d_S ? d_S[m] : nullptr, d_theta ? d_theta[m] : nullptr, d_psi ? d_psi[m] : nullptr};
        for (const float *p : ptrs)
            if (p && ((uintptr_t)p & 15)) return fail(c, CYRSOXS_ERR_INVALID_ARG, "material %d: array not 16-byte aligned", m);
    }
    for (int m = 0; m < c->n_mat; ++m) {
        c->mp.phi[m] = d_phi[m];
        c->mp.S[m] = d_S ? d_S[m] : nullptr;
        c->mp.theta[m] = d_theta ? d_theta[m] : nullptr;
        c->mp.psi[m] = d_psi ? d_psi[m] : nullptr;
    }
    c->streamed = false;
    if (!c->owned_morph.empty()) {
        // device copies left by an earlier cyrsoxs_set_morphology_host / _aos (cudaFree waits for the work that reads them)
        DeviceGuard guard(c->device);
        for (void *p : c->owned_morph) cudaFree(p);
        c->owned_morph.clear();
        c->plan_eb = 0;                      // the energy batch was planned with less free memory
    }
    note_null_pattern(c);
    c->have_morph = true;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_morphology_host(cyrsoxs_ctx *c, const float *const *h_phi, const float *const *h_S,
                                           const float *const *h_theta, const float *const *h_psi, void *cuda_stream)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    cyrsoxs_status st = check_morph_tables(c, h_phi, h_S, h_theta, h_psi);
    if (st != CYRSOXS_OK) return st;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    DeviceGuard guard(c->device);
    // an earlier run on another stream may still be reading the buffers this call overwrites
    if (c->ran && s != c->last_stream) CUDA_TRY(c, cudaStreamWaitEvent(s, c->ev_run_done, 0));
    const size_t bytes = sizeof(float) * (size_t)c->Nx * c->Ny * c->Nz;
    // count arrays, (re)allocate owned buffers
    std::vector<const float *> src;
    for (int m = 0; m < c->n_mat; ++m) {
        src.push_back(h_phi[m]);
        src.push_back(h_S ? h_S[m] : nullptr);
        src.push_back(h_theta ? h_theta[m] : nullptr);
        src.push_back(h_psi ? h_psi[m] : nullptr);
    }
    size_t need = 0;
    for (const float *p : src) need += p ? 1 : 0;
    if (c->owned_morph.size() != need) {
        for (void *p : c->owned_morph) cudaFree(p);
        c->owned_morph.clear();
        for (size_t i = 0; i < need; ++i) {
            void *d = nullptr;
            cudaError_t e = cudaMalloc(&d, bytes);
            if (e != cudaSuccess) {
                cudaGetLastError();
                for (void *p : c->owned_morph) cudaFree(p);
                c->owned_morph.clear();
                c->have_morph = false;
                return fail(c, CYRSOXS_ERR_OOM, "cudaMalloc(morphology, %zu bytes): %s", bytes, cudaGetErrorString(e));
            }
            c->owned_morph.push_back(d);
        }
    }
    size_t slot = 0;
    const float *dptr[4 * MAX_MAT];
    for (size_t i = 0; i < src.size(); ++i) {
        dptr[i] = nullptr;
        if (!src[i]) continue;
        void *d = c->owned_morph[slot++];
        CUDA_TRY(c, cudaMemcpyAsync(d, src[i], bytes, cudaMemcpyHostToDevice, s));
        dptr[i] = (const float *)d;
    }
    for (int m = 0; m < c->n_mat; ++m) {
        c->mp.phi[m] = dptr[4 * m]; c->mp.S[m] = dptr[4 * m + 1];
        c->mp.theta[m] = dptr[4 * m + 2]; c->mp.psi[m] = dptr[4 * m + 3];
    }
    c->streamed = false;
    note_null_pattern(c);
    c->have_morph = true;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_morphology_streamed(cyrsoxs_ctx *c, const float *const *h_phi, const float *const *h_S,
                                               const float *const *h_theta, const float *const *h_psi, int materials_per_group)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    cyrsoxs_status st = check_morph_tables(c, h_phi, h_S, h_theta, h_psi);
    if (st != CYRSOXS_OK) return st;
    if (materials_per_group < 1) return fail(c, CYRSOXS_ERR_INVALID_ARG, "materials_per_group must be >= 1");
    for (int m = 0; m < c->n_mat; ++m) {
        c->host_mp.phi[m] = h_phi[m];
        c->host_mp.S[m] = h_S ? h_S[m] : nullptr;
        c->host_mp.theta[m] = h_theta ? h_theta[m] : nullptr;
        c->host_mp.psi[m] = h_psi ? h_psi[m] : nullptr;
        c->mp.phi[m] = c->mp.S[m] = c->mp.theta[m] = c->mp.psi[m] = nullptr;
    }
    c->host_mp.n_mat = c->n_mat;
    c->streamed = true;
    c->stream_group = std::min(materials_per_group, c->n_mat);
    {
        DeviceGuard guard(c->device);
        for (void *p : c->owned_morph) cudaFree(p);
        c->owned_morph.clear();
    }
    c->plan_dirty = true;
    note_null_pattern(c);
    c->have_morph = true;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_morphology_aos(cyrsoxs_ctx *c, const float *d_real4, void *cuda_stream)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (!d_real4) return fail(c, CYRSOXS_ERR_INVALID_ARG, "morphology array is NULL");
    if ((uintptr_t)d_real4 & 15) return fail(c, CYRSOXS_ERR_INVALID_ARG, "morphology array not 16-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(c->device);
    if (c->ran && st != c->last_stream) CUDA_TRY(c, cudaStreamWaitEvent(st, c->ev_run_done, 0));
    const size_t n = (size_t)c->Nx * c->Ny * c->Nz, bytes = sizeof(float) * n;
    const size_t need = 4 * (size_t)c->n_mat;
    if (c->owned_morph.size() != need) {
        for (void *p : c->owned_morph) cudaFree(p);
        c->owned_morph.clear();
        for (size_t i = 0; i < need; ++i) {
            void *d = nullptr;
            cudaError_t e = cudaMalloc(&d, bytes);
            if (e != cudaSuccess) {
                cudaGetLastError();
                for (void *p : c->owned_morph) cudaFree(p);
                c->owned_morph.clear();
                c->have_morph = false;
                return fail(c, CYRSOXS_ERR_OOM, "cudaMalloc(morphology, %zu bytes): %s", bytes, cudaGetErrorString(e));
            }
            c->owned_morph.push_back(d);
        }
    }
    cyrsoxs_status s = ensure(c, c->red, sizeof(unsigned int) * MAX_MAT);
    if (s != CYRSOXS_OK) return s;
    CUDA_TRY(c, cudaMemsetAsync(c->red.p, 0, sizeof(unsigned int) * MAX_MAT, st));
    const int grid = std::min<long long>(((long long)n + 255) / 256, 8LL * c->n_sm);
    for (int m = 0; m < c->n_mat; ++m) {
        float *a[4];
        for (int j = 0; j < 4; ++j) a[j] = (float *)c->owned_morph[4 * m + j];
        k_aos_to_soa<<<grid, 256, 0, st>>>((const float4 *)d_real4 + (size_t)m * n, a[0], a[1], a[2], a[3], n,
                                           (unsigned int *)c->red.p + m);
        CUDA_TRY(c, cudaGetLastError());
    }
    unsigned int bits[MAX_MAT];
    CUDA_TRY(c, cudaMemcpyAsync(bits, c->red.p, sizeof(unsigned int) * c->n_mat, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaStreamSynchronize(st));
    for (int m = 0; m < c->n_mat; ++m) {
        const bool aligned = bits[m] != 0;
        c->mp.phi[m] = (const float *)c->owned_morph[4 * m];
        c->mp.S[m] = aligned ? (const float *)c->owned_morph[4 * m + 1] : nullptr;
        c->mp.theta[m] = aligned ? (const float *)c->owned_morph[4 * m + 2] : nullptr;
        c->mp.psi[m] = aligned ? (const float *)c->owned_morph[4 * m + 3] : nullptr;
    }
    c->streamed = false;
    note_null_pattern(c);
    c->have_morph = true;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_optical_constants(cyrsoxs_ctx *c, int n_energy, const double *energies_eV,
                                             const float *delta_par, const float *beta_par,
                                             const float *delta_perp, const float *beta_perp)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (n_energy < 1 || !energies_eV || !delta_par || !beta_par || !delta_perp || !beta_perp)
        return fail(c, CYRSOXS_ERR_INVALID_ARG, "optical constants: NULL table or n_energy < 1");
    for (int e = 0; e < n_energy; ++e)
        if (!(energies_eV[e] > 0.0) || !isfinite(energies_eV[e]))
            return fail(c, CYRSOXS_ERR_INVALID_ARG, "energy %d is not positive", e);
    const int M = c->n_mat;
    c->nE = n_energy;
    c->energies.assign(energies_eV, energies_eV + n_energy);
    c->k.resize(n_energy);
    c->coef.resize((size_t)n_energy * M * 6);
    typedef std::complex<double> cd;
    const double inv4pi = 1.0 / (4.0 * kPi);
    for (int e = 0; e < n_energy; ++e) {
        const double lambda = kHcEvNm / energies_eV[e];
        c->k[e] = (2.0 * kPi) / lambda;
        for (int m = 0; m < M; ++m) {
            const size_t i = (size_t)e * M + m;
            // n - 1 = -delta + i beta; n^2 - 1 = (n - 1)(n + 1): nothing of size 1 cancels
            const cd npar(-(double)delta_par[i], (double)beta_par[i]), nperp(-(double)delta_perp[i], (double)beta_perp[i]);
            const cd niso = (npar + 2.0 * nperp) / 3.0;
            const cd a = nperp * (nperp + 2.0), b = (npar - nperp) * (npar + nperp + 2.0), cc = niso * (niso + 2.0);
            // a - c = (n_perp - n_iso)(n_perp + n_iso), again without cancellation
            const cd amc = (nperp - niso) * (nperp + niso + 2.0);
            const cd Cc = cc * inv4pi, Ca = amc * inv4pi, Cb = b * inv4pi;
            (void)a;
            float *o = &c->coef[i * 6];
            o[0] = (float)Cc.real(); o[1] = (float)Cc.imag();
            o[2] = (float)Ca.real(); o[3] = (float)Ca.imag();
            o[4] = (float)Cb.real(); o[5] = (float)Cb.imag();
        }
    }
    {
        // reach of the valid disk in x pixels, see k_rotate_avg
        c->reach2.resize(n_energy);
        const double rho = (double)c->Nx / (double)c->Ny;
        for (int e = 0; e < n_energy; ++e) {
            const double r = c->k[e] / c->dqx + sqrt(1.0 + rho * rho) + 1.0;
            c->reach2[e] = (float)(r * r * 1.0001);
        }
    }
    // the device copies are refreshed by the next cyrsoxs_run, on its stream (a run still executing keeps its tables)
    c->have_optics = true;
    c->optics_dirty = true;
    c->plan_dirty = true;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_angles(cyrsoxs_ctx *c, double start_deg, double step_deg, double end_deg)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (!isfinite(start_deg) || !isfinite(step_deg) || !isfinite(end_deg))
        return fail(c, CYRSOXS_ERR_INVALID_ARG, "angles must be finite");
    int n;
    if (start_deg == end_deg) n = 1;
    else {
        if (step_deg == 0.0) return fail(c, CYRSOXS_ERR_INVALID_ARG, "angle step is 0 with start != end");
        double q = floor((end_deg - start_deg) / step_deg + 1e-9);
        if (q < 0.0) return fail(c, CYRSOXS_ERR_INVALID_ARG, "(end - start)/step is negative");
        if (q + 1.0 > (double)kMaxAngles) return fail(c, CYRSOXS_ERR_INVALID_ARG, "more than %d angles", kMaxAngles);
        n = (int)q + 1;
    }
    c->nA = n;
    c->cs.resize(n);
    std::vector<float4> &csf = c->csf;
    csf.resize(n);
    for (int i = 0; i < n; ++i) {
        const double zeta = start_deg + (double)i * step_deg;
        const double zr = zeta * (kPi / 180.0);
        double C = cos(zr), S = sin(zr);
        if (fabs(C) < 1e-15) C = 0.0;
        if (fabs(S) < 1e-15) S = 0.0;
        c->cs[i] = make_double2(C, S);
        csf[i] = make_float4((float)(C * C), (float)(S * S), (float)(2.0 * C * S), 0.f);
    }
    c->have_angles = true;
    c->angles_dirty = true;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_ewald(cyrsoxs_ctx *c, cyrsoxs_ewald mode)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (mode != CYRSOXS_EWALD_NEAREST && mode != CYRSOXS_EWALD_TRILINEAR) return fail(c, CYRSOXS_ERR_INVALID_ARG, "unknown Ewald mode");
    c->ewald = mode;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_algorithm(cyrsoxs_ctx *c, cyrsoxs_algorithm alg)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (alg != CYRSOXS_ALG_AUTO && alg != CYRSOXS_ALG_PER_ENERGY && alg != CYRSOXS_ALG_SPECTRAL_BASIS)
        return fail(c, CYRSOXS_ERR_INVALID_ARG, "unknown algorithm");
    if (alg != c->alg) c->spectra_ready = false;     // spectra of a run under another setting are not handed to run_energies
    c->alg = alg;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_counts_output(cyrsoxs_ctx *c, unsigned int *d_counts)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    c->d_counts = d_counts;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_profiling(cyrsoxs_ctx *c, int enabled)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    c->profiling = enabled ? 1 : 0;
    return CYRSOXS_OK;
}

int cyrsoxs_num_angles(const cyrsoxs_ctx *c) { return c && c->have_angles ? c->nA : 0; }

// phases: 1 = the energy-independent spectra (SPECTRAL_BASIS), 2 = the energies of the range; cyrsoxs_run does both
enum { PHASE_SPECTRA = 1, PHASE_ENERGIES = 2 };

static cyrsoxs_status run_body(cyrsoxs_ctx *c, void *cuda_stream, float *out, int phases);

// A run that fails partway may already have enqueued work on `cuda_stream` that uses the shared workspace: mark the end of
// that partial work too, so that the next run on ANOTHER stream still waits for it (ev_run_done pairs with last_stream).
static cyrsoxs_status run_impl(cyrsoxs_ctx *c, void *cuda_stream, float *out, int phases)
{
    const cyrsoxs_status s = run_body(c, cuda_stream, out, phases);
    if (s != CYRSOXS_OK && c && c->ev_run_done && c->last_stream == (cudaStream_t)cuda_stream) {
        DeviceGuard guard(c->device);
        if (cudaEventRecord(c->ev_run_done, c->last_stream) == cudaSuccess) c->ran = true;
        else cudaGetLastError();
    }
    return s;
}

static cyrsoxs_status run_body(cyrsoxs_ctx *c, void *cuda_stream, float *out, int phases)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if ((phases & PHASE_ENERGIES) && !out) return fail(c, CYRSOXS_ERR_INVALID_ARG, "out is NULL");
    if (!c->have_morph || !c->have_optics || !c->have_angles)
        return fail(c, CYRSOXS_ERR_NOT_READY, "run needs morphology, optical constants and angles (missing:%s%s%s)",
                    c->have_morph ? "" : " morphology", c->have_optics ? "" : " optical-constants", c->have_angles ? "" : " angles");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(c->device);
    if (!c->ev_run_done) CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_run_done, cudaEventDisableTiming));
    // the workspace and the device tables are shared by consecutive runs: a run on another stream waits for the last one
    if (c->ran && st != c->last_stream) CUDA_TRY(c, cudaStreamWaitEvent(st, c->ev_run_done, 0));
    c->last_stream = st;             // from here on everything this call enqueues is on st (run_impl marks its end, also on failure)

    // where does `out` live?
    bool out_on_host = false;
    if (phases & PHASE_ENERGIES) {
        cudaPointerAttributes pa{};
        cudaError_t pe = cudaPointerGetAttributes(&pa, out);
        if (pe != cudaSuccess) { cudaGetLastError(); return fail(c, CYRSOXS_ERR_INVALID_ARG, "out: %s", cudaGetErrorString(pe)); }
        out_on_host = pa.type == cudaMemoryTypeHost;
        if (pa.type != cudaMemoryTypeHost && pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)
            return fail(c, CYRSOXS_ERR_INVALID_ARG, "out must be device memory or pinned host memory");
    }
    // the energies this call processes (cyrsoxs_set_energy_range); windows and tables always cover all of them
    const int e_first = c->e_count < 0 ? 0 : c->e_first, nE_run = c->e_count < 0 ? c->nE : c->e_count;
    if (e_first < 0 || nE_run < 1 || e_first + nE_run > c->nE)
        return fail(c, CYRSOXS_ERR_INVALID_ARG, "energy range [%d, %d) is not inside the %d energies set", e_first, e_first + nE_run, c->nE);

    // programmatic dependent launch for small runs only (see launch_pdl)
    c->pdl = (double)c->Nx * c->Ny * c->Nz <= (double)(1 << 23) && (double)c->Nx * c->Ny * c->nE <= (double)(1 << 24);
#ifdef CYRSOXS_TUNING
    if (const char *e = getenv("CYRSOXS_PDL")) c->pdl = atoi(e) != 0;
#endif
    cyrsoxs_status s;
    if ((s = upload_tables(c, st)) != CYRSOXS_OK) return s;
    if (c->plan_dirty && (s = build_basis_plan(c, st)) != CYRSOXS_OK) return s;
    // AUTO: the basis needs n_pack complex transforms per run, PER_ENERGY 5 per energy; a basis transform
    // (register-first x pass, real fields) costs about half of a PER_ENERGY one (measured on cfg3: 0.31 ms
    // per pack against 0.6 ms per field), hence the factor 2
    int alg = c->alg;
    if (alg == CYRSOXS_ALG_AUTO)
        alg = (c->streamed || !is_pow2(c->Nx) || 2 * NCHI * c->nE >= c->n_pack) ? CYRSOXS_ALG_SPECTRAL_BASIS : CYRSOXS_ALG_PER_ENERGY;
    if (!is_pow2(c->Nx) && alg != CYRSOXS_ALG_SPECTRAL_BASIS)
        return fail(c, CYRSOXS_ERR_NOT_IMPLEMENTED, "Nx that is not a power of two needs CYRSOXS_ALG_SPECTRAL_BASIS (or AUTO)");
    if (c->streamed && alg != CYRSOXS_ALG_SPECTRAL_BASIS)
        return fail(c, CYRSOXS_ERR_NOT_IMPLEMENTED, "a streamed morphology needs CYRSOXS_ALG_SPECTRAL_BASIS (or AUTO)");
    const bool spectral = alg == CYRSOXS_ALG_SPECTRAL_BASIS;

    // plan: windows for the largest k, energy batch from the free memory
    double kmax = *std::max_element(c->k.begin(), c->k.end());
    Window wx, wy, wz;
    int pitch;
    windows_for(c, kmax, wx, wy, wz, pitch, spectral);
    const size_t npix = (size_t)c->Nx * c->Ny;
    const size_t F1 = spectral ? (size_t)c->n_pack : (size_t)NCHI;
    const size_t a1 = F1 * c->Nz * c->Ny * pitch, a2 = c->Nz > 1 ? F1 * wz.W * c->Ny * pitch : 0, a3 = F1 * wz.W * wy.W * pitch;
    c->A3_pack_bytes = sizeof(float2) * (size_t)wz.W * wy.W * pitch;
    const size_t per_img = sizeof(float4) * npix + (out_on_host ? 2 * sizeof(float) * npix : 0);
    const size_t per_e = spectral ? per_img : sizeof(float2) * (a1 + a2 + a3) + per_img;
    const size_t stage_bytes = c->streamed ? 2 * (size_t)c->stream_group * 4 * sizeof(float) * (size_t)c->Nx * c->Ny * c->Nz : 0;
    const size_t fixed = (spectral ? sizeof(float2) * (a1 + a2 + a3) : 0) + stage_bytes;
    // The energy batch depends on the free device memory; cudaMemGetInfo is slow, so the batch is
    // re-planned only when what it depends on has changed since the last run.
    if (c->shard_parts > 1 && (!spectral || c->streamed))
        return fail(c, CYRSOXS_ERR_NOT_IMPLEMENTED, "a spectra shard needs CYRSOXS_ALG_SPECTRAL_BASIS (or AUTO) and a resident morphology");
    const unsigned long long plan_key = (unsigned long long)nE_run * 8 + (spectral ? 4 : 0) + (out_on_host ? 2 : 0) + 1;
    int eb = c->plan_eb;
    if (plan_key != c->plan_key || fixed != c->plan_fixed || per_e != c->plan_per_e || eb < 1) {
        size_t free_b = 0, total_b = 0;
        CUDA_TRY(c, cudaMemGetInfo(&free_b, &total_b));
        const size_t have = c->A1.cap + c->A2.cap + c->A3.cap + c->img.cap + c->stage_out[0].cap + c->stage_out[1].cap
                            + c->stage_morph[0].cap + c->stage_morph[1].cap;
        const size_t budget = (size_t)((double)(free_b + have) * 0.85);
        if (fixed + per_e > budget)
            return fail(c, CYRSOXS_ERR_OOM, "workspace of %.1f GB does not fit in %.1f GB of free device memory",
                        (double)(fixed + per_e) / 1e9, (double)budget / 1e9);
        eb = (int)std::min<size_t>((size_t)nE_run, std::max<size_t>(1, (budget - fixed) / per_e));
        if (!spectral) {
            // ~2 GiB of fields per batch is plenty of parallelism
            const size_t target = (size_t)1 << 31;
            eb = (int)std::max<size_t>(1, std::min<size_t>((size_t)eb, std::max<size_t>(1, target / (sizeof(float2) * a1))));
        } else {
            const size_t target = (size_t)1 << 32;
            eb = (int)std::max<size_t>(1, std::min<size_t>((size_t)eb, std::max<size_t>(1, target / per_img)));
        }
        eb = std::min(eb, 256);
        if (eb < nE_run && eb >= 8) eb = eb / 8 * 8;              // whole image groups in all but the last batch
        c->plan_key = plan_key; c->plan_fixed = fixed; c->plan_per_e = per_e; c->plan_eb = eb;
    }
    c->eg = choose_eg(eb);
    const size_t eb_pad = (size_t)(eb + c->eg - 1) / c->eg * c->eg;
    const size_t mult = spectral ? 1 : (size_t)eb;
    if ((s = ensure(c, c->A1, sizeof(float2) * a1 * mult)) != CYRSOXS_OK) return s;
    if (a2 && (s = ensure(c, c->A2, sizeof(float2) * a2 * mult)) != CYRSOXS_OK) return s;
    if ((s = ensure(c, c->A3, sizeof(float2) * a3 * mult)) != CYRSOXS_OK) return s;
    if ((s = ensure(c, c->img, sizeof(float4) * npix * eb_pad)) != CYRSOXS_OK) return s;
    if (out_on_host) {
        for (int i = 0; i < 2; ++i)
            if ((s = ensure(c, c->stage_out[i], sizeof(float) * npix * eb)) != CYRSOXS_OK) return s;
        if (!c->copy_stream) CUDA_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            if (!c->ev_batch[i]) CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_batch[i], cudaEventDisableTiming));
            if (!c->ev_copy[i]) CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_copy[i], cudaEventDisableTiming));
        }
    }

    clear_prof(c);
    memset(&c->stats, 0, sizeof c->stats);
    c->stats.algorithm = alg;
    c->stats.n_energy = nE_run; c->stats.n_angles = c->nA; c->stats.energy_batch = eb;
    c->stats.workspace_bytes = (double)(c->A1.cap + c->A2.cap + c->A3.cap + c->img.cap + c->stage_out[0].cap + c->stage_out[1].cap);
    c->last_stream = st;

    // spectra_ready means "A3 holds the basis spectra of the current configuration": only the spectral path sets it, and a
    // PER_ENERGY run, whose phase 1 is empty and whose phase 2 fills A1..A3 with per-energy chi spectra, takes it away
    if (!spectral)
        c->spectra_ready = false;
    else if (phases & PHASE_SPECTRA) {
        c->spectra_ready = false;
        if ((s = run_basis_spectra(c, st, wx, wy, wz, pitch)) != CYRSOXS_OK) return s;
        c->spectra_ready = true;
    } else if (!c->spectra_ready)
        return fail(c, CYRSOXS_ERR_NOT_READY, "cyrsoxs_run_energies needs cyrsoxs_run_spectra first (after the last change of morphology, constants, shard or algorithm)");

    int nb = 0;
    for (int e0 = e_first; (phases & PHASE_ENERGIES) && e0 < e_first + nE_run; e0 += eb, ++nb) {
        const int n = std::min(eb, e_first + nE_run - e0);
        // `out` and the counts buffer hold the energies of the range only
        unsigned int *cnt = c->d_counts ? c->d_counts + (size_t)(e0 - e_first) * npix : nullptr;
        float *dst = out + (size_t)(e0 - e_first) * npix;
        const int slot = nb & 1;
        if (out_on_host) {
            // the staging slot is free once the copy issued two batches ago has finished
            if (nb >= 2) CUDA_TRY(c, cudaStreamWaitEvent(st, c->ev_copy[slot], 0));
            dst = (float *)c->stage_out[slot].p;
        }
        s = spectral ? run_batch_spectral(c, st, e0, n, wx, wy, wz, pitch, dst, cnt) : run_batch_per_energy(c, st, e0, n, dst, cnt);
        if (s != CYRSOXS_OK) return s;
        if (out_on_host) {
            CUDA_TRY(c, cudaEventRecord(c->ev_batch[slot], st));
            CUDA_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->ev_batch[slot], 0));
            CUDA_TRY(c, cudaMemcpyAsync(out + (size_t)(e0 - e_first) * npix, dst, sizeof(float) * npix * n, cudaMemcpyDeviceToHost, c->copy_stream));
            CUDA_TRY(c, cudaEventRecord(c->ev_copy[slot], c->copy_stream));
        }
        c->last_batch_e = n;
    }
    if (out_on_host) {
        // `out` is complete when `st` reaches this point
        for (int i = 0; i < std::min(nb, 2); ++i) CUDA_TRY(c, cudaStreamWaitEvent(st, c->ev_copy[i], 0));
    }
    CUDA_TRY(c, cudaEventRecord(c->ev_run_done, st));
    c->ran = true;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_run(cyrsoxs_ctx *c, void *cuda_stream, float *out) { return run_impl(c, cuda_stream, out, PHASE_SPECTRA | PHASE_ENERGIES); }

cyrsoxs_status cyrsoxs_run_spectra(cyrsoxs_ctx *c, void *cuda_stream) { return run_impl(c, cuda_stream, nullptr, PHASE_SPECTRA); }

cyrsoxs_status cyrsoxs_run_energies(cyrsoxs_ctx *c, void *cuda_stream, float *out) { return run_impl(c, cuda_stream, out, PHASE_ENERGIES); }

cyrsoxs_status cyrsoxs_set_spectra_shard(cyrsoxs_ctx *c, int part, int n_parts)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (n_parts < 1 || n_parts > c->n_mat || part < 0 || part >= n_parts)
        return fail(c, CYRSOXS_ERR_INVALID_ARG, "spectra shard: 1 <= n_parts <= n_mat (%d) and 0 <= part < n_parts", c->n_mat);
    c->shard_part = part; c->shard_parts = n_parts;
    c->plan_dirty = true;
    c->spectra_ready = false;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_set_energy_range(cyrsoxs_ctx *c, int first, int count)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (count >= 0 && (first < 0 || count < 1)) return fail(c, CYRSOXS_ERR_INVALID_ARG, "energy range: first >= 0 and count >= 1 (or count < 0 for all)");
    c->e_first = count < 0 ? 0 : first; c->e_count = count < 0 ? -1 : count;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_get_spectra(cyrsoxs_ctx *c, void **d_spectra, unsigned long long *pack_bytes, int *n_pack)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (!c->spectra_ready || !c->A3.p) return fail(c, CYRSOXS_ERR_NOT_READY, "no spectra yet: call cyrsoxs_run_spectra first");
    if (d_spectra) *d_spectra = c->A3.p;
    if (pack_bytes) *pack_bytes = (unsigned long long)c->A3_pack_bytes;
    if (n_pack) *n_pack = c->n_pack;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_get_spectra_part(cyrsoxs_ctx *c, int part, int *first_pack, int *n_pack)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (!c->spectra_ready) return fail(c, CYRSOXS_ERR_NOT_READY, "no spectra yet: call cyrsoxs_run_spectra first");
    if (part < 0 || part >= (int)c->part_pack0.size()) return fail(c, CYRSOXS_ERR_INVALID_ARG, "no such part");
    if (first_pack) *first_pack = c->part_pack0[part];
    if (n_pack) *n_pack = c->part_npack[part];
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_get_stats(cyrsoxs_ctx *c, cyrsoxs_stats *stats)
{
    if (!c || !stats) return CYRSOXS_ERR_INVALID_ARG;
    if (c->profiling && !c->prof_events.empty()) {
        DeviceGuard guard(c->device);
        CUDA_TRY(c, cudaStreamSynchronize(c->last_stream));
        for (int i = 0; i < CYRSOXS_N_STAGES; ++i) c->stats.stage_ms[i] = 0.f;
        for (size_t i = 0; i < c->prof_stage.size(); ++i) {
            float ms = 0.f;
            CUDA_TRY(c, cudaEventElapsedTime(&ms, c->prof_events[2 * i], c->prof_events[2 * i + 1]));
            c->stats.stage_ms[c->prof_stage[i]] += ms;
        }
    }
    *stats = c->stats;
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_reduce(cyrsoxs_ctx *c, void *cuda_stream, const float *d_images, const unsigned int *d_counts,
                              int n_energy, int n_bins, double sector_half_width_deg, float *d_I, float *d_A, float *d_isi)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (!d_images || !d_I) return fail(c, CYRSOXS_ERR_INVALID_ARG, "reduce: images or I output is NULL");
    if (n_energy < 1 || n_bins < 1 || n_bins > 4096) return fail(c, CYRSOXS_ERR_INVALID_ARG, "reduce: n_energy >= 1 and 1 <= n_bins <= 4096");
    if (!(sector_half_width_deg > 0.0) || !(sector_half_width_deg <= 45.0))
        return fail(c, CYRSOXS_ERR_INVALID_ARG, "reduce: sector half width must be in (0, 45] degrees");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(c->device);
    const size_t nb = (size_t)n_energy * 3 * n_bins;
    const size_t bytes = sizeof(double) * nb + sizeof(double) * n_energy + sizeof(unsigned int) * nb;
    cyrsoxs_status s = ensure(c, c->red, bytes);
    if (s != CYRSOXS_OK) return s;
    CUDA_TRY(c, cudaMemsetAsync(c->red.p, 0, bytes, st));
    ReduceParams p{};
    p.Nx = c->Nx; p.Ny = c->Ny; p.n_bins = n_bins;
    p.rho = (double)c->Nx / (double)c->Ny;
    p.tan_w = tan(sector_half_width_deg * (kPi / 180.0));
    p.img = d_images; p.cnt = d_counts;
    p.acc = (double *)c->red.p; p.total = p.acc + nb; p.num = (unsigned int *)(p.total + n_energy);
    // enough CTAs to fill the machine, at least 4 rows each so the shared-memory bins are amortised
    const int want = std::max(1, 4 * c->n_sm / n_energy);
    p.rows_per_cta = std::max(4, (c->Ny + want - 1) / want);
    const dim3 grid((c->Ny + p.rows_per_cta - 1) / p.rows_per_cta, n_energy);
    const size_t smem = (size_t)3 * n_bins * (sizeof(double) + sizeof(unsigned int));
    if (smem > 48 * 1024)
        if (cyrsoxs_status a = allow_smem(c, k_reduce_accumulate, (size_t)3 * 4096 * 12)) return a;
    k_reduce_accumulate<<<grid, 256, smem, st>>>(p);
    CUDA_TRY(c, cudaGetLastError());
    const int tot = n_energy * n_bins;
    k_reduce_finalize<<<(tot + 255) / 256, 256, 0, st>>>(n_energy, n_bins, p.acc, p.num, p.total, c->dqx * c->dqy, d_I, d_A, d_isi);
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

} // extern "C"

// ---- cyrsoxs_reduce_static: the reduction's scratch without cudaMalloc ------------------------------------------------
// The per-bin sums, pixel counts and per-energy totals that k_reduce_accumulate hands to k_reduce_finalize normally sit
// in c->red (cudaMalloc'ed on first use).  Callers that cannot allocate (HBM already owned by another pool, or no
// tolerance for cudaMalloc's device-wide synchronisation; see include/cyrsoxs.h) get the same two kernels pointed at this
// array instead.  It is part of the library's device image: every GPU that loads the library holds
// CYRSOXS_REDUCE_STATIC_BYTES for it until the process exits.
//
// In HOST code the name g_reduce_static is only a handle for the runtime's symbol calls, NOT a device address: giving
// `g_reduce_static` (or &g_reduce_static[0]) to a kernel faults, or on systems where the GPU can reach host memory quietly
// works on the wrong bytes.  The address each device uses comes from cudaGetSymbolAddress, asked once per device with that
// device current (reduce_static_address below) and then passed to the kernels like any other pointer.
static __device__ __align__(256) unsigned char g_reduce_static[CYRSOXS_REDUCE_STATIC_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_reduce_static_mutex;                    // contexts of different host threads may reach the table together
void *g_reduce_static_ptr[kMaxDevices] = {};          // device address of g_reduce_static on device i, nullptr = not asked yet

// Device address of g_reduce_static on the context's device, which the caller has made current.  The first call per
// device asks the runtime (this may load the library's device code there: keep it out of stream captures); later calls
// read the table.
cyrsoxs_status reduce_static_address(cyrsoxs_ctx *c, void **out)
{
    if (c->device < 0 || c->device >= kMaxDevices) return fail(c, CYRSOXS_ERR_INVALID_ARG, "reduce_static: device index %d beyond %d", c->device, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_reduce_static_mutex);
    if (!g_reduce_static_ptr[c->device]) {
        int cur = -1;
        CUDA_TRY(c, cudaGetDevice(&cur));
        if (cur != c->device) return fail(c, CYRSOXS_ERR_CUDA, "reduce_static: device %d could not be made current (current: %d)", c->device, cur);
        void *ptr = nullptr;
        CUDA_TRY(c, cudaGetSymbolAddress(&ptr, g_reduce_static));
        if (!ptr) return fail(c, CYRSOXS_ERR_CUDA, "reduce_static: cudaGetSymbolAddress returned a null address");
        g_reduce_static_ptr[c->device] = ptr;
    }
    *out = g_reduce_static_ptr[c->device];
    return CYRSOXS_OK;
}

} // namespace

extern "C" {

cyrsoxs_status cyrsoxs_reduce_static(cyrsoxs_ctx *c, void *cuda_stream, const float *d_images, const unsigned int *d_counts,
                                     int n_energy, int n_bins, double sector_half_width_deg, float *d_I, float *d_A, float *d_isi)
{
    if (!c) return CYRSOXS_ERR_INVALID_ARG;
    if (!d_images || !d_I) return fail(c, CYRSOXS_ERR_INVALID_ARG, "reduce_static: images or I output is NULL");
    if (n_energy < 1 || n_bins < 1) return fail(c, CYRSOXS_ERR_INVALID_ARG, "reduce_static: n_energy >= 1 and n_bins >= 1");
    if (n_bins > CYRSOXS_REDUCE_STATIC_MAX_BINS || n_energy > CYRSOXS_REDUCE_STATIC_MAX_ENERGIES
        || (long long)n_energy * n_bins > CYRSOXS_REDUCE_STATIC_MAX_CELLS)
        return fail(c, CYRSOXS_ERR_INVALID_ARG,
                    "reduce_static: %d energies x %d bins exceed the fixed scratch (at most %d bins, %d energies, %d energies x bins); "
                    "use cyrsoxs_reduce, which allocates", n_energy, n_bins, CYRSOXS_REDUCE_STATIC_MAX_BINS,
                    CYRSOXS_REDUCE_STATIC_MAX_ENERGIES, CYRSOXS_REDUCE_STATIC_MAX_CELLS);
    if (!(sector_half_width_deg > 0.0) || !(sector_half_width_deg <= 45.0))
        return fail(c, CYRSOXS_ERR_INVALID_ARG, "reduce_static: sector half width must be in (0, 45] degrees");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(c->device);
    void *scratch = nullptr;
    if (cyrsoxs_status s = reduce_static_address(c, &scratch)) return s;
    // same layout as cyrsoxs_reduce inside its buffer: [e][3][bins] double sums, [e] double totals, [e][3][bins] counts
    const size_t nb = (size_t)n_energy * 3 * n_bins;
    const size_t bytes = sizeof(double) * nb + sizeof(double) * n_energy + sizeof(unsigned int) * nb;
    static_assert(sizeof(double) * 3 * CYRSOXS_REDUCE_STATIC_MAX_CELLS + sizeof(double) * CYRSOXS_REDUCE_STATIC_MAX_ENERGIES
                      + sizeof(unsigned int) * 3 * CYRSOXS_REDUCE_STATIC_MAX_CELLS == CYRSOXS_REDUCE_STATIC_BYTES,
                  "the limits of include/cyrsoxs.h size the array");
    // the array still holds the previous call's sums (any context, any stream): the kernels add into it, so zero what
    // this call uses, stream-ordered before them
    CUDA_TRY(c, cudaMemsetAsync(scratch, 0, bytes, st));
    ReduceParams p{};
    p.Nx = c->Nx; p.Ny = c->Ny; p.n_bins = n_bins;
    p.rho = (double)c->Nx / (double)c->Ny;
    p.tan_w = tan(sector_half_width_deg * (kPi / 180.0));
    p.img = d_images; p.cnt = d_counts;
    p.acc = (double *)scratch; p.total = p.acc + nb; p.num = (unsigned int *)(p.total + n_energy);
    const int want = std::max(1, 4 * c->n_sm / n_energy);
    p.rows_per_cta = std::max(4, (c->Ny + want - 1) / want);
    const dim3 grid((c->Ny + p.rows_per_cta - 1) / p.rows_per_cta, n_energy);
    // 36 KB at the bin limit: below the 48 KB a kernel may use without raising its attribute
    const size_t smem = (size_t)3 * n_bins * (sizeof(double) + sizeof(unsigned int));
    static_assert((size_t)3 * CYRSOXS_REDUCE_STATIC_MAX_BINS * 12 <= 48 * 1024, "bin limit keeps the default shared-memory size");
    k_reduce_accumulate<<<grid, 256, smem, st>>>(p);
    CUDA_TRY(c, cudaGetLastError());
    const int tot = n_energy * n_bins;
    k_reduce_finalize<<<(tot + 255) / 256, 256, 0, st>>>(n_energy, n_bins, p.acc, p.num, p.total, c->dqx * c->dqy, d_I, d_A, d_isi);
    CUDA_TRY(c, cudaGetLastError());
    return CYRSOXS_OK;
}

cyrsoxs_status cyrsoxs_debug_fetch_images(cyrsoxs_ctx *c, int e_in_batch, float *d_dst)
{
    if (!c || !d_dst) return CYRSOXS_ERR_INVALID_ARG;
    if (!c->img.p || e_in_batch < 0 || e_in_batch >= c->last_batch_e) return fail(c, CYRSOXS_ERR_INVALID_ARG, "no such image");
    DeviceGuard guard(c->device);
    const size_t npix = (size_t)c->Nx * c->Ny;
    const int eg = c->eg;
    const float4 *src = (const float4 *)c->img.p + (size_t)(e_in_batch / eg) * npix * eg + e_in_batch % eg;
    CUDA_TRY(c, cudaMemcpy2DAsync(d_dst, sizeof(float4), src, sizeof(float4) * eg, sizeof(float4), npix,
                                  cudaMemcpyDeviceToDevice, c->last_stream));
    return CYRSOXS_OK;
}

} // extern "C"
