/*
 * cyrsoxs.h -- C ABI of libcyrsoxs, the B200 (sm_100a) forward-simulation hot path of
 * CyRSoXS (arXiv 2209.13121).  Citations: P:n = PAPER.md line n; "DESIGN 3-Ax" = the
 * reading of the paper fixed in DESIGN.md section 3.
 *
 * What one cyrsoxs_run computes (Algorithm 1), for every energy E_i and every
 * in-plane E-field angle zeta of E_Angle[start, increment, end]:
 *   1. induced polarization per voxel, Eq. 2-5:
 *        p = (1/4pi) sum_m phi_m [ S_m ((n_perp^2-1) e + (n_par^2-n_perp^2)(d_m.e) d_m)
 *                                  + (1-S_m)(n_iso^2-1) e ],
 *        e = (cos zeta, sin zeta, 0), d = (cos psi sin theta, sin psi sin theta, cos theta),
 *        n = 1 - delta + i beta, n_iso = (n_par + 2 n_perp)/3;
 *   2. p~ = FFT(p), Eq. 6, forward, unnormalised, origin at voxel 0;
 *   3. X = |k^2 (I - r r^T) p~|^2 on the Ewald sphere, Eq. 7-8:
 *        q_z = sqrt(k^2 - q_x^2 - q_y^2) - k, k = 2 pi E / 1239.84197 nm^-1, real q_z only,
 *        X taken at the nearest k_z bin or interpolated linearly between the two neighbours;
 *   4. the image of each angle rotated back by -zeta about q = 0 (bilinear) and averaged over
 *      the angles with per-pixel valid counts.
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback.
 *
 * Layouts.  Voxel (x, y, z) of a morphology array is element x + Nx (y + Ny z) (x fastest).
 * Output pixel (iy, ix) of energy i is out[(i Ny + iy) Nx + ix] and corresponds to
 * (q_x, q_y) = ((ix - Nx/2) dq_x, (iy - Ny/2) dq_y), dq = 2 pi / (N voxel_nm); q = 0 sits at
 * (Ny/2, Nx/2).  Pixels that are valid at no angle are written as 0.0f.
 *
 * Threading: a context is not thread-safe; use one context per host thread / per GPU.
 * Every function returns a status and never throws, aborts or prints.
 */
#ifndef CYRSOXS_H
#define CYRSOXS_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cyrsoxs_ctx cyrsoxs_ctx; /* opaque; created and destroyed by the library */

typedef enum {
    CYRSOXS_OK = 0,
    CYRSOXS_ERR_INVALID_ARG = 1,     /* bad size, NULL where not allowed, bad enum, bad angle spec */
    CYRSOXS_ERR_NOT_READY = 2,       /* run before all of: morphology, optical constants, angles    */
    CYRSOXS_ERR_CUDA = 3,            /* a CUDA call failed; cyrsoxs_last_error has the CUDA string  */
    CYRSOXS_ERR_OOM = 4,             /* device (or pinned host) memory exhausted                    */
    CYRSOXS_ERR_NOT_IMPLEMENTED = 5
} cyrsoxs_status;

typedef enum {
    CYRSOXS_EWALD_NEAREST = 0,       /* X at k_z = floor(q_z/dq_z + 0.5) (north_star; not in the paper) */
    CYRSOXS_EWALD_TRILINEAR = 1      /* X interpolated linearly between floor and floor+1      */
} cyrsoxs_ewald;

/* How the per-energy work is organised; all choices give the same images (tests check it).
 *   PER_ENERGY      the paper's order with p linear in e (north_star): per energy the five
 *                   distinct entries of the susceptibility tensor chi (xx, xy, xz, yy, yz; p for
 *                   e = x is its first column, for e = y its second) are formed per voxel,
 *                   transformed, and projected.  Kept as the reference organisation (closest to
 *                   Algorithm 1) and for runs with one energy and many aligned materials; its x
 *                   pass uses the first-generation FFT core and is not the tuned path.
 *   SPECTRAL_BASIS  p is also linear in the optical constants: the energy-independent real
 *                   fields phi, phi S, phi S d_i d_j are transformed once per run and every
 *                   energy only combines their spectra on its Ewald shell (DESIGN 7.0).
 *   AUTO            SPECTRAL_BASIS unless the basis needs more than 10 complex transforms per
 *                   energy of the run (n_pack > 10 n_energy: one energy, many aligned materials). */
typedef enum {
    CYRSOXS_ALG_AUTO = 0,
    CYRSOXS_ALG_PER_ENERGY = 1,
    CYRSOXS_ALG_SPECTRAL_BASIS = 2
} cyrsoxs_algorithm;

/* Stage ids of cyrsoxs_stats (stage_launches, stage_bytes, stage_ms). */
typedef enum {
    CYRSOXS_STAGE_XPASS = 0,   /* polarization (or basis fields) fused with the FFT along x  */
    CYRSOXS_STAGE_ZPASS = 1,   /* FFT along z, pruned to the k_z planes the Ewald shells touch */
    CYRSOXS_STAGE_YPASS = 2,   /* FFT along y, pruned to |k_y| <= k/dq_y                       */
    CYRSOXS_STAGE_EWALD = 3,   /* Ewald gather + (I - r r^T) + |.|^2 -> (I_xx, I_yy, I_xy, valid) */
    CYRSOXS_STAGE_ROTATE = 4,  /* rotate back by -zeta, accumulate over angles, divide by counts */
    CYRSOXS_N_STAGES = 5
} cyrsoxs_stage;

typedef struct {
    int algorithm;                 /* cyrsoxs_algorithm actually used by the last run           */
    int n_energy, n_angles;
    int energy_batch;              /* energies processed per kernel launch group                */
    long long kernel_launches;     /* kernels launched by the last run                          */
    long long stage_launches[CYRSOXS_N_STAGES];
    double stage_bytes[CYRSOXS_N_STAGES];   /* algorithmic HBM bytes per stage, whole run (DESIGN 8) */
    float stage_ms[CYRSOXS_N_STAGES];       /* device time per stage, whole run; 0 unless profiling  */
    double workspace_bytes;        /* device scratch owned by the context                       */
} cyrsoxs_stats;

/* Creates a context for an Nx x Ny x Nz voxel model with n_mat materials and cubic voxels of
 * edge voxel_nm ("voxels are considered perfect cubes").  4 <= Nx <= 2048, 2 <= Ny <= 2048,
 * 1 <= Nz <= 2048.  Powers of two take the FFT kernels (the paper recommends them laterally); an
 * axis of any other length (the paper uses Nz = 63) is transformed by the definition of Eq. 6
 * evaluated at the bins the Ewald step can reach (a pruned direct DFT, O(N W) per line: a functional
 * path for thin films and odd lateral sizes, not a tuned FFT -- measured on B200: Nz = 63 costs 3.6 x
 * Nz = 64 at 1024 x 1024, a 1000 x 600 x 1 film 4 ms, a 1000 x 1000 x 64 volume 120 x the 1024 x 1024 x 64
 * one; pad large volumes laterally to a power of two where possible).  Nx that is not a power of two needs
 * CYRSOXS_ALG_SPECTRAL_BASIS (AUTO picks it; PER_ENERGY returns NOT_IMPLEMENTED at run).
 * 1 <= n_mat <= 32, voxel_nm > 0 (else INVALID_ARG); voxel_nm is a double because the detector grid dq = 2 pi / (N voxel_nm)
 * and with it every validity decision is formed in double (DESIGN 3-A11).  Uses the current CUDA device.  *out is NULL on
 * failure. */
cyrsoxs_status cyrsoxs_create(int Nx, int Ny, int Nz, int n_mat, double voxel_nm, cyrsoxs_ctx **out);

/* Morphology (memory model P:199-203): for each material m four DEVICE arrays of
 * Nx*Ny*Nz float32: volume fraction phi (the paper's v_frac), alignment S, and the director's
 * polar angle theta (from +z) and azimuth psi (from +x), radians.  d_phi etc. are HOST arrays
 * of n_mat device pointers.  d_S[m], d_theta[m], d_psi[m] may all be NULL together for an
 * isotropic material (S == 0); d_S, d_theta, d_psi themselves may be NULL if every material
 * is isotropic.  Pointers are BORROWED: the caller keeps the arrays alive and unmodified until
 * every run that uses them has completed.  Arrays must be 16-byte aligned.  The library does
 * not check sum_m phi_m = 1 (neither does the paper's code) nor clamp S.
 * Angle range: SPECTRAL_BASIS forms sin and cos of theta and psi with the hardware approximation
 * (about 5e-7 absolute) and no extended range reduction, which holds for |angle| up to a few pi
 * (tests cover [-3 pi, 3 pi]); beyond that the error of each director component grows by about
 * 6e-8 |angle| (3e-6 at 50 rad: images then agree with a double-precision evaluation to about
 * 1e-4 instead of 1e-5).  Wrap angles into [-pi, pi] on the caller's side if they can be large.
 * PER_ENERGY uses sincosf, accurate at any magnitude. */
cyrsoxs_status cyrsoxs_set_morphology(cyrsoxs_ctx *ctx, const float *const *d_phi,
                                      const float *const *d_S, const float *const *d_theta,
                                      const float *const *d_psi);

/* Same, from HOST arrays (pinned or pageable): copied into device buffers owned by the context
 * with cudaMemcpyAsync on `cuda_stream` (the paper's one-off M_GPU <- M_CPU, Alg. 1 line 1,
 * P:220).  The host arrays must stay valid until that stream reaches the end of the copy. */
cyrsoxs_status cyrsoxs_set_morphology_host(cyrsoxs_ctx *ctx, const float *const *h_phi,
                                           const float *const *h_S, const float *const *h_theta,
                                           const float *const *h_psi, void *cuda_stream);

/* Same, from the paper's own layout (Fig. 3): one DEVICE array of n_mat * Nx*Ny*Nz
 * Real4 = float4 entries, voxels first and materials second (entry m*N + i), each entry
 * (v_frac, s, Euler-phi, theta) = (phi, S, psi, theta) in this header's names.  The array is
 * de-interleaved on `cuda_stream` into structure-of-arrays buffers owned by the context (the
 * kernels read those; d_real4 is not referenced after the stream passes this call).  A material
 * whose S is 0 in every voxel is detected and treated as isotropic.  16-byte alignment required.
 * This call synchronises `cuda_stream` once (to read back the per-material max |S|). */
cyrsoxs_status cyrsoxs_set_morphology_aos(cyrsoxs_ctx *ctx, const float *d_real4, void *cuda_stream);

/* Memory-minimising variant (the idea of the paper's Algorithm 2/3: the morphology is
 * only needed while the polarization precursor is formed, so it is streamed through the device
 * instead of kept there).  The four tables are HOST arrays of n_mat HOST pointers (as in
 * cyrsoxs_set_morphology_host, PINNED memory for the copies to overlap) that are BORROWED: they
 * must stay valid and unmodified across every later cyrsoxs_run.  Each run uploads the materials
 * `materials_per_group` (>= 1) at a time into a double-buffered device staging area of
 * 2 * materials_per_group * 16 bytes per voxel on an internal copy stream, while the previous
 * group's fields are transformed; the device never holds more of the morphology than that.
 * The energy-independent spectra of SPECTRAL_BASIS play the role of the paper's N_t (they are
 * formed once per run, not once per energy); CYRSOXS_ALG_PER_ENERGY is refused in this mode
 * (NOT_IMPLEMENTED at cyrsoxs_run).  Results equal the resident mode's within rounding (fields
 * are paired inside a group, so the pairing can differ). */
cyrsoxs_status cyrsoxs_set_morphology_streamed(cyrsoxs_ctx *ctx, const float *const *h_phi,
                                               const float *const *h_S, const float *const *h_theta,
                                               const float *const *h_psi, int materials_per_group);

/* Energy list and the material library: HOST arrays, copied.  energies_eV has
 * n_energy entries (> 0); the four tables are [n_energy][n_mat] float32 with
 * n_par = 1 - delta_par + i beta_par, n_perp likewise.  The complex coefficients
 * n_perp^2 - 1, n_par^2 - n_perp^2, n_iso^2 - 1 are formed here in double as (n-1)(n+1) and
 * rounded once to float32. */
cyrsoxs_status cyrsoxs_set_optical_constants(cyrsoxs_ctx *ctx, int n_energy, const double *energies_eV,
                                             const float *delta_par, const float *beta_par,
                                             const float *delta_perp, const float *beta_perp);

/* E_Angle[start, increment, end] in degrees: zeta_n = start + n step for
 * n = 0 .. floor((end - start)/step + 1e-9); start == end gives one angle.  INVALID_ARG for
 * step == 0 with start != end, for (end - start)/step < 0, or for more than 4096 angles. */
cyrsoxs_status cyrsoxs_set_angles(cyrsoxs_ctx *ctx, double start_deg, double step_deg, double end_deg);

/* Ewald interpolation along q_z; default CYRSOXS_EWALD_TRILINEAR (the paper's). */
cyrsoxs_status cyrsoxs_set_ewald(cyrsoxs_ctx *ctx, cyrsoxs_ewald mode);

/* Work organisation; default CYRSOXS_ALG_AUTO. */
cyrsoxs_status cyrsoxs_set_algorithm(cyrsoxs_ctx *ctx, cyrsoxs_algorithm alg);

/* Optional second output of cyrsoxs_run: per-pixel number of angles that contributed,
 * n_energy*Ny*Nx unsigned ints in DEVICE memory, same layout as out.  NULL (default) disables. */
cyrsoxs_status cyrsoxs_set_counts_output(cyrsoxs_ctx *ctx, unsigned int *d_counts);

/* When enabled, each run brackets every stage with CUDA events and cyrsoxs_get_stats reports
 * stage_ms (this serialises the internal streams a little; keep it off for throughput runs). */
cyrsoxs_status cyrsoxs_set_profiling(cyrsoxs_ctx *ctx, int enabled);

/* Runs the whole path for all energies and angles.  All work is enqueued on `cuda_stream`
 * (a cudaStream_t; NULL = the legacy default stream) and on internal streams fenced to it by
 * events; the call returns without synchronising, and `out` is complete when `cuda_stream`
 * reaches the point after the call.  `out` is n_energy*Ny*Nx float32 in DEVICE memory, or in
 * PINNED HOST memory (then each energy batch's images are copied back asynchronously while
 * the next batch computes, "the averaged result is transferred from GPU to CPU").
 * Scratch is allocated on first use and kept by the context (ERR_OOM if it does not fit). */
cyrsoxs_status cyrsoxs_run(cyrsoxs_ctx *ctx, void *cuda_stream, float *out);

/* Number of angles currently configured (0 before cyrsoxs_set_angles). */
int cyrsoxs_num_angles(const cyrsoxs_ctx *ctx);

/* ---- Two-phase run and spectra shards (multi-GPU, DESIGN 11) ------------------------------------------------------
 * With CYRSOXS_ALG_SPECTRAL_BASIS a run is (1) the energy-independent spectra of the basis fields -- almost all of the
 * device time on large volumes -- and (2) per energy the Ewald gather and the rotate/average step.  Energies shard over
 * GPUs without communication, but phase 1 would then be repeated by every GPU; it shards over MATERIALS instead:
 *
 *   cyrsoxs_set_spectra_shard(ctx, part, n_parts)   the materials are cut into n_parts contiguous groups of about equal
 *       field count (7 fields per aligned material, 1 per isotropic one; 1 <= n_parts <= n_mat); this context transforms
 *       group `part` only.  The fields of a group are paired among themselves (an odd count is padded), so the pack layout
 *       depends on n_parts, not on `part`: every GPU that sets the same n_parts has the same layout.  Needs a resident
 *       morphology and SPECTRAL_BASIS (else NOT_IMPLEMENTED at run).  (0, 1) restores the unsharded layout.  A shard
 *       divides the transform WORK, not the workspace: every context still holds the x- and z-pass buffers and the
 *       spectra buffer for all packs (the other parts' spectra are copied into the latter).
 *   cyrsoxs_set_energy_range(ctx, first, count)     phase 2 (and cyrsoxs_run) processes energies [first, first + count)
 *       of the tables given to cyrsoxs_set_optical_constants; `out` and the counts buffer then hold `count` images.  The
 *       spectral windows are always sized for ALL energies of the tables, so GPUs with different ranges share one layout.
 *       count < 0: all energies (default).
 *   cyrsoxs_run_spectra(ctx, stream)                phase 1 for this context's part, enqueued on `stream`.
 *   cyrsoxs_get_spectra(ctx, &d_ptr, &pack_bytes, &n_pack)   the context-owned DEVICE buffer of the pruned spectra,
 *       n_pack consecutive blocks of pack_bytes ([k_z window][k_y window][x pitch] complex64 each); valid until the next
 *       change of sizes, constants or shard.  cyrsoxs_get_spectra_part(ctx, part, &first_pack, &n_pack) names the blocks
 *       a part owns.  The caller copies the other parts' blocks in (NCCL broadcast / all_gather, or cudaMemcpyPeer),
 *       ordered after phase 1 and before phase 2 on the streams it uses.
 *   cyrsoxs_run_energies(ctx, stream, out)          phase 2 on whatever the spectra buffer holds (NOT_READY unless
 *       cyrsoxs_run_spectra ran, under SPECTRAL_BASIS, after the last change of morphology, constants, shard or
 *       algorithm, and no PER_ENERGY run has overwritten the buffer since).
 * cyrsoxs_run is phase 1 followed by phase 2; with a shard of more than one part it produces images from this part's
 * materials only, so sharded callers use the two calls.  PER_ENERGY: phase 1 is empty, phase 2 does everything. */
cyrsoxs_status cyrsoxs_set_spectra_shard(cyrsoxs_ctx *ctx, int part, int n_parts);
cyrsoxs_status cyrsoxs_set_energy_range(cyrsoxs_ctx *ctx, int first, int count);
cyrsoxs_status cyrsoxs_run_spectra(cyrsoxs_ctx *ctx, void *cuda_stream);
cyrsoxs_status cyrsoxs_get_spectra(cyrsoxs_ctx *ctx, void **d_spectra, unsigned long long *pack_bytes, int *n_pack);
cyrsoxs_status cyrsoxs_get_spectra_part(cyrsoxs_ctx *ctx, int part, int *first_pack, int *n_pack);
cyrsoxs_status cyrsoxs_run_energies(cyrsoxs_ctx *ctx, void *cuda_stream, float *out);

/* Counters of the last run (see cyrsoxs_stats).  Synchronises `cuda_stream` of that run if
 * profiling is enabled. */
cyrsoxs_status cyrsoxs_get_stats(cyrsoxs_ctx *ctx, cyrsoxs_stats *stats);

/* 1-D reductions of finished images (the quantities of the paper's
 * validation figures: azimuthal average I(|q|) Fig. 5b/8b P:387 P:415, scattering anisotropy
 * Fig. 15, integrated scattering intensity Fig. 6 / Eq. 10).  The paper gives no
 * binning rule; DESIGN.md 12 fixes one.  For each of the n_energy images d_images[e][Ny][Nx]
 * (DEVICE, e.g. the `out` of cyrsoxs_run) and with u = ix - Nx/2, v = (iy - Ny/2) Nx/Ny:
 *   radial bin b = floor(sqrt(u^2 + v^2) + 1/2), kept if b < n_bins (|q| = b dq_x);
 *   only pixels with d_counts[e][iy][ix] > 0 take part (d_counts NULL: all pixels);
 *   d_I[e][b]    mean over the bin's pixels (0 if none);
 *   d_A[e][b]    (I_para - I_perp)/(I_para + I_perp), sector means over the bin's pixels within
 *                sector_half_width_deg of the q_x axis (para: the E-field axis after the
 *                rotate-back step) resp. of the q_y axis; 0 if a sector is empty;
 *   d_isi[e]     dq_x dq_y times the sum over ALL valid pixels of the image.
 * All outputs are float32 in DEVICE memory (d_A and d_isi may be NULL); sums are accumulated in
 * double.  1 <= n_bins <= 4096, 0 < sector_half_width_deg <= 45.  Enqueued on cuda_stream. */
cyrsoxs_status cyrsoxs_reduce(cyrsoxs_ctx *ctx, void *cuda_stream, const float *d_images,
                              const unsigned int *d_counts, int n_energy, int n_bins,
                              double sector_half_width_deg, float *d_I, float *d_A, float *d_isi);

/* cyrsoxs_reduce for callers that must not allocate device memory.  Same arguments, same kernels and same results as
 * cyrsoxs_reduce, but the per-bin sums the kernels need between their two
 * launches live in a fixed array compiled into the library instead of a cudaMalloc'ed, context-owned buffer.
 *
 * Who needs it.  cudaMalloc can fail or hurt in a process that is otherwise healthy: (1) a host application (a PyTorch
 * caching allocator, a reconstruction or fitting service at the beamline) that has already claimed the whole of HBM for
 * its own pool, so any further cudaMalloc returns out-of-memory although the pool could have lent the bytes; (2) a
 * live-analysis loop that reduces every detector frame as it arrives and cannot accept the device-wide synchronisation
 * cudaMalloc and cudaFree imply, which stalls every other stream of the process for the length of the call.  Such
 * callers create the context once at start-up, while allocating is still possible (cyrsoxs_create uploads a few KB of
 * twiddle tables), and from then on use this call only: it performs no cudaMalloc, no cudaFree and calls no library
 * routine that allocates; images and outputs are the caller's.
 *
 * Limits (INVALID_ARG with an explanatory cyrsoxs_last_error beyond them; use cyrsoxs_reduce for larger reductions):
 *   1 <= n_bins <= CYRSOXS_REDUCE_STATIC_MAX_BINS, 1 <= n_energy <= CYRSOXS_REDUCE_STATIC_MAX_ENERGIES,
 *   n_energy * n_bins <= CYRSOXS_REDUCE_STATIC_MAX_CELLS.
 * The array is CYRSOXS_REDUCE_STATIC_BYTES (about 1.2 MB) of device memory on EVERY GPU on which the process uses this
 * library, from the moment the library's code is loaded there until the process exits, whether or not this call is made.
 *
 * First call per device.  The first call on each GPU looks up the device address of the array (cudaGetSymbolAddress with
 * that GPU current) and caches it; make that first call during start-up, outside any stream capture.  Later calls only
 * enqueue one memset and two kernels on `cuda_stream`.
 *
 * Sharing.  There is ONE array per GPU, shared by every context and every call in the process, and it keeps what the last
 * call left in it.  Each call therefore zeroes the part it uses, on `cuda_stream`, before its kernels run.  Two calls whose
 * GPU work can overlap (different streams without an event between them, or two host threads) race on the array and
 * produce garbage in both outputs: order them on one stream or with events.  Calls do not overlap with cyrsoxs_reduce's
 * scratch, which is a different buffer. */
#define CYRSOXS_REDUCE_STATIC_MAX_BINS 1024
#define CYRSOXS_REDUCE_STATIC_MAX_ENERGIES 1024
#define CYRSOXS_REDUCE_STATIC_MAX_CELLS 32768
#define CYRSOXS_REDUCE_STATIC_BYTES (3 * 12 * CYRSOXS_REDUCE_STATIC_MAX_CELLS + 8 * CYRSOXS_REDUCE_STATIC_MAX_ENERGIES)
cyrsoxs_status cyrsoxs_reduce_static(cyrsoxs_ctx *ctx, void *cuda_stream, const float *d_images,
                                     const unsigned int *d_counts, int n_energy, int n_bins,
                                     double sector_half_width_deg, float *d_I, float *d_A, float *d_isi);

/* Test hook, not part of the contract: copies the per-energy Ewald images of the LAST energy
 * batch of the last run, as float4 (I_xx, I_yy, I_xy, valid) per pixel, for batch-local energy
 * index `e_in_batch`, into d_dst (Ny*Nx*4 floats, device).  Enqueued on the run's stream. */
cyrsoxs_status cyrsoxs_debug_fetch_images(cyrsoxs_ctx *ctx, int e_in_batch, float *d_dst);

/* Human-readable description of the last error of this context ("" if none).  The string is
 * owned by the context and valid until the next call on it.  Accepts NULL (returns a static
 * string describing a creation failure). */
const char *cyrsoxs_last_error(const cyrsoxs_ctx *ctx);

/* Frees the context and its scratch; borrowed morphology arrays are left alone.  NULL is ok. */
void cyrsoxs_destroy(cyrsoxs_ctx *ctx);

/* Library version string, e.g. "cyrsoxs-b200 0.1 (sm_100a)". */
const char *cyrsoxs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CYRSOXS_H */
