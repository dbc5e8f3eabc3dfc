/* apic.h - C ABI of libapic: B200-native APIC closed-form reconstruction.
 *
 * The operation is the per-tile reconstruction of arXiv 2407.20469 (§2.3, lines 64-135,
 * Fig. 2 at line 70): a stack of intensity images I_i taken under NA-matching and darkfield LED
 * illumination is turned into an aberration-corrected complex field on an upsampled grid plus the
 * tile's recovered pupil.  Steps, each executed by hand-written sm_100a kernels:
 *   S0     background flag (BASELINE.json item 5)
 *   S1-S5  Kramers-Kronig field retrieval, Eq. 4-7
 *   S6     aberration extraction from phase differences in overlaps, Eq. 8-10,
 *          in a Noll-Zernike basis, weighted normal equations + Cholesky (BASELINE.json item 3)
 *   S7     correction + stitching
 *   S8-S10 darkfield extension, Eq. 11-13, matrix-free CGLS on C u = d
 *   S10    zero-padded inverse transform to the u*N grid, pupil output
 * Readings of the silent / garbled points are DESIGN.md §3 (R1-R23 of SURVEY.md §8(c)).
 *
 * Conventions: images and fields are row-major [y][x], x fastest; the spatial origin is pixel
 * (0,0); raw pixel m maps to output pixel u*m; spectra are normalised so that DC = spatial mean.
 * A blank object (amplitude 1, phase 0) gives I = 1 in every NA-matching image and a field = 1.
 *
 * All functions return 0 (APIC_OK) on success and a negative apic_error otherwise.  No exceptions
 * cross the boundary and there is no CPU fallback: if no CUDA device is usable the calls fail with
 * APIC_ECUDA.  A plan belongs to the CUDA device that was current at apic_plan_create: its tables,
 * workspace and kernel attributes live there, every call on the plan makes that device current for
 * its duration (and restores the caller's), and streams passed to it must belong to that device.
 * Plans on different devices may coexist in one process.  The only process-wide state is the
 * per-device twiddle cache of the two test entries apic_fft2d / apic_fft2d_xy (mutex-protected) and
 * the thread-local error strings.  A plan is not thread-safe; use one plan per stream.
 */
#ifndef APIC_H_
#define APIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct apic_plan apic_plan; /* opaque; owns all device tables and the workspace */

typedef enum {
  APIC_OK = 0,
  APIC_EINVAL = -1,   /* bad parameter / geometry (see apic_plan_create) */
  APIC_ECUDA = -2,    /* a CUDA runtime call failed (apic_last_cuda_error gives the text) */
  APIC_ENOMEM = -3,   /* host or device allocation failed */
  APIC_EBATCH = -4,   /* batch outside 1..max_batch */
  APIC_ESCRATCH = -5  /* problem larger than the scratch built into the library (apic_reassemble_static) */
} apic_error;

/* Per-tile status written to d_status. */
enum {
  APIC_TILE_OK = 0,
  APIC_TILE_BACKGROUND = 1, /* skipped by the background criterion; outputs are zero          */
  APIC_TILE_BAD_INPUT = 2,  /* a non-finite input pixel (or scale); outputs are zero.  Negative
                               values are NOT bad input: read noise produces them, the log clamps
                               them (intensity_floor, R6) and the darkfield right-hand
                               side uses them as they are (B5)                        */
  APIC_TILE_SOLVE_FAILED = 3 /* weighted phase residual of the aberration fit > 1 rad RMS (or
                                non-finite); outputs are still written                        */
};

typedef struct {
  int tile_n;            /* N: raw tile side, 64 | 128 | 256 | 512                               */
  int upsample;          /* u: 1..4, output grid is (u*N)^2                                       */
  double wavelength_um;  /* lambda                                                              */
  double pixel_um;       /* effective pixel = camera pitch / magnification         */
  double na_obj;         /* objective NA                                                        */
  int n_bright;          /* number of NA-matching LEDs (>= 3)                                    */
  const double* k_bright;/* host, [n_bright][2] (kx,ky) in cycles/um, |k| = NA/lambda*/
  int n_dark;            /* number of darkfield LEDs (may be 0)                                  */
  const double* k_dark;  /* host, [n_dark][2], |k| > NA/lambda; NULL if n_dark == 0               */
  int n_zernike;         /* number of fitted Zernike terms (1..64)                               */
  const int* noll;       /* host, [n_zernike] distinct Noll indices, each >= 4 (piston and tilts
                            are the exact null space of Eq. 10; R9)                    */
  int kk_pad;            /* 1 or 2 (2: tile_n <= 256).  The log of Eq. 5 is not band-limited; with 2
                            every NA-matching image is Fourier-interpolated to the 2N grid before
                            the log and the KK chain runs there, which removes the aliasing floor
                            of the retrieved field (2e-4 -> 4e-9 on config 0; R7) at 4x
                            the transform work of S1-S5                                          */
  int refine_iters;      /* re-wrapped refinements of the aberration fit (R11); 0..16   */
  int df_iters;          /* maximum CGLS iterations per darkfield LED (>= 1)                      */
  float df_tol;          /* CGLS stops when ||C^H r|| <= df_tol * ||C^H d||; 0 = run df_iters.
                            (There is no df_solver field: SURVEY.md 8(b) listed one for a dense
                            Cholesky alternative; that route was measured at ~60x the cost of the
                            matrix-free CG - DESIGN.md section 5, "The dense route" - and is not
                            built, so a selector would have one legal value.)                    */
  float intensity_floor; /* I <- max(I, floor * mean(I)) before the log (R6)            */
  int bg_mode;           /* 0 off | 1: mean(I_bright) >= bg_threshold | 2: var/mean^2 <= thr      */
  float bg_threshold;
  int max_batch;         /* apic_reconstruct accepts 1..max_batch tiles; workspace is sized for
                            min(max_batch, internal chunk)                                       */
  int chunk_tiles;       /* tiles per internal pass; 0 = chosen by the library: one tile per SM
                            (148 on B200: teams of two CTAs) for the reduced-grid darkfield
                            kernels (N = 256, whose working set is ~0.3 MB per tile), otherwise as many tiles as
                            keep the full-grid darkfield working set (1.7 N^2 complex64 per tile)
                            inside half of the device's L2 (queried), clamped to 8..512          */
  int df_mode;           /* darkfield scheduler.  Every mode runs one launch per pass that covers
                            all darkfield LEDs; a thread-block cluster (team) owns a tile and
                            meets at cluster barriers between phases.  At N = 256 modes 0, 4, 5, 6
                            run the CG mat-vecs on per-LED reduced cyclic grids (DESIGN.md
                            section 5); other N run mode 3 whatever is asked.
                            0 = default: df_wide.cu in df_mgrid.cu's shape (teams of 256-thread
                                CTAs, 128 registers, 2 CTAs per SM) with the p_M strips and Q
                                masks parked in shared memory and the CG vectors distributed
                                over the team.
                            3 = the team kernel on the full N x N grid (cross-check of the
                                reduced grids).
                            4 = strips staged by the async proxy (cp.async.bulk + mbarrier,
                                strip-major scratch), df_tma.cu.
                            5 = pairs of 1024-thread CTAs at 64 registers (four strip groups per
                                CTA); LEDs whose grid fits run the CG loop decimated 2 x 2 with
                                the classes resident in shared memory (two cluster barriers per
                                iteration), df_wide.cu.
                            6 = df_mgrid.cu, the round-1 kernel (redundant CG vectors, plain
                                loads).  Measured on config 2: 0 is the
                                fastest, 4-6 are kept as named, parity-tested alternatives     */
  int df_team;           /* CTAs per tile: 1, 2, 4 or 8 (anything else is APIC_EINVAL); 0 = chosen
                            from the pass size (as many as the pass leaves resident CTA slots
                            for; the automatic choice may also take 5, which cannot be asked for) */
  int df_order;          /* order of the darkfield extension (PAPER.md:135 states none).  0 = one
                            LED after the other by ascending |kappa|, ties by input order; a bin
                            belongs to the first LED that solves it (reading R15, the default).
                            1 = ring-wise (reading R15b): every LED of a ring (equal |kappa|) is
                            solved against the known set as it stands when the ring starts, bins
                            solved by several LEDs of the ring get the mean of their solutions,
                            the known set grows once per ring                                   */
} apic_params;

/* Fills *p with the defaults (kk_pad 1, refine_iters 3, df_iters 48, df_tol 1e-4, floor 1e-6,
 * bg off, max_batch 64); the caller then sets the geometry fields. */
void apic_params_default(apic_params* p);

/* Builds every geometry-only table on the host in fp64 (disc masks, half-plane weights of Eq. 5,
 * overlap sets S_il of Eq. 8 and the rows of Eq. 10, darkfield sets P/U/Q of Eq. 13, Zernike
 * tables, FFT twiddles), uploads them to the current CUDA device and allocates the workspace.
 * The arrays inside *p are copied.  APIC_EINVAL if: N not in {64,128,256,512}; u outside 1..4;
 * an NA-matching LED with | |kappa_i| - R | > 0.5 bin; the synthetic aperture does not fit the raw
 * grid (max|kappa| + R >= N/2 - 1); a darkfield LED whose unknown fraction exceeds 42 %
 * or whose linear region Q is empty; a Noll index < 4 or repeated; kk_pad not 1 or 2; fewer than one
 * overlapping pair. */
int apic_plan_create(const apic_params* p, apic_plan** out);
int apic_plan_destroy(apic_plan* plan);

typedef struct {
  int tile_n, upsample, out_n;    /* out_n = u*N                                                */
  int n_bright, n_dark, n_zernike;
  int n_pairs;                    /* overlapping NA-matching pairs (Eq. 8)                       */
  int n_rows, n_grad_rows;        /* rows of Eq. 10 / of the gradient-domain initialisation      */
  int n_union;                    /* bins covered by the NA-matching discs                       */
  int n_known;                    /* bins of the final extended spectrum                         */
  int n_dark_used;                /* darkfield LEDs with a non-empty unknown set                 */
  int max_unknown, max_equations; /* max |U_i|, max |Q_i|                                        */
  int chunk_tiles;                /* tiles processed per internal pass                          */
  size_t table_bytes, workspace_bytes;
  double radius_bins;             /* R = NA*N*dx/lambda                                          */
} apic_plan_info_t;
int apic_plan_info(const apic_plan* plan, apic_plan_info_t* info);

/* The same geometry numbers computed on the host only (no CUDA device is touched; table_bytes,
 * workspace_bytes and chunk_tiles are 0).  If led / n_unknown / n_equations are non-NULL they
 * receive up to `cap` darkfield index-set sizes in processing order.  Used by the CPU tests. */
int apic_geometry_info(const apic_params* p, apic_plan_info_t* info, int* led, int* n_unknown,
                       int* n_equations, int cap);
/* Host only: the reduced cyclic grid (mx, my) chosen for each used darkfield LED, in processing
 * order (alias-free iff mx, my exceed the extent of U - P - Q per axis). */
int apic_geometry_dark_grids(const apic_params* p, int* mx, int* my, int cap);

/* Darkfield index-set sizes in processing order (ascending |kappa|, ties by input order):
 * led[k] = input index, n_unknown[k] = |U|, n_equations[k] = |Q|.  Arrays hold n_dark_used ints. */
int apic_plan_dark_sets(const apic_plan* plan, int* led, int* n_unknown, int* n_equations);

/* The whole hot path for `batch` tiles.  Every pointer is a DEVICE pointer owned by the caller;
 * all work is enqueued on `cuda_stream` (a cudaStream_t, NULL = legacy default stream).  With
 * bg_mode == 0 the call returns without synchronising; with bg_mode != 0 it synchronises the
 * stream once, after the background pass, to read the number of tiles left to reconstruct.
 *   d_intensity [batch][n_bright+n_dark][N][N] float, NA-matching images first, LED order = plan
 *               order, common radiometric units (R17)
 *   d_field     [batch][uN][uN] complex64 as (re,im) float pairs
 *   d_zernike   [batch][n_zernike] float, rad, Noll-normalised, order = plan's noll[]
 *   d_pupil     [batch][N][N] complex64, 1[|k|<=R] exp(j phi_hat(k)), centred (bin 0 at N/2); or NULL
 *   d_status    [batch] int32, APIC_TILE_*
 */
int apic_reconstruct(apic_plan* plan, const float* d_intensity, int batch, float* d_field,
                     float* d_zernike, float* d_pupil, int32_t* d_status, void* cuda_stream);

/* Same call with HOST buffers (pinned or pageable): copies the inputs to the device, runs
 * apic_reconstruct, copies the results back and synchronises before returning.  Batches of >= 32
 * tiles are cut into min(8, batch / 16) equal sub-batches (each >= 16 tiles) that alternate between two
 * workspace sets (the second is allocated on first use) and two compute streams, with uploads and downloads on two
 * copy streams, so that copies in both directions overlap the kernels.  h_pupil may be NULL. */
int apic_reconstruct_host(apic_plan* plan, const float* h_intensity, int batch, float* h_field,
                          float* h_zernike, float* h_pupil, int32_t* h_status, void* cuda_stream);

/* The same reconstruction from raw camera counts (BASELINE.json config 2: "uint16 raw converted to
 * fp32"; exposures differ between NA-matching and darkfield frames,
 * PAPER.md:199):
 *   d_raw    [batch][n_bright+n_dark][N][N] uint16, same order as d_intensity
 *   d_scale  [batch][n_bright+n_dark] float: intensity = count * scale (1 / (gain * exposure) of
 *            that frame, so that all frames are in common radiometric units, R17)
 * The conversion float(count) * scale (one fp32 multiply) is fused into the loads of the three steps
 * that read images - S0 statistics, S1 log-intensity, S8 darkfield right-hand side - so no fp32 copy
 * of the counts exists and the input bytes read from HBM are halved; the results equal
 * apic_reconstruct on float(count) * scale bit for bit (tested, incl. the background decision).
 * A non-finite scale makes the tile APIC_TILE_BAD_INPUT.  Other arguments as apic_reconstruct. */
int apic_reconstruct_u16(apic_plan* plan, const uint16_t* d_raw, const float* d_scale, int batch,
                         float* d_field, float* d_zernike, float* d_pupil, int32_t* d_status,
                         void* cuda_stream);
/* ... and with HOST buffers (half the host-to-device bytes of apic_reconstruct_host). */
int apic_reconstruct_host_u16(apic_plan* plan, const uint16_t* h_raw, const float* h_scale, int batch,
                              float* h_field, float* h_zernike, float* h_pupil, int32_t* h_status,
                              void* cuda_stream);

/* Streaming form of the host entries, for a sequence of batches (a slide is thousands of tiles,
 * PAPER.md:177-179): apic_submit_host[_u16] enqueues the upload, the kernels and the download of one
 * batch in pipeline slot `slot` (0 or 1) and returns without waiting; apic_wait_host(plan, slot)
 * blocks until that batch's results are in its host buffers and returns its status.  With one
 * batch in flight per slot the upload of batch k+1 and the download of batch k-1 overlap the
 * kernels of batch k, so a long sequence runs at max(upload, kernels, download) per batch instead of
 * their sum.  The host buffers should be pinned (pageable memory makes the copies synchronous) and
 * must stay valid and untouched until the wait returns; a slot must be waited for before it is
 * submitted to again (a busy slot is waited for implicitly).  Results are the bits of
 * apic_reconstruct on the same inputs.  With bg_mode != 0 a submit blocks until the batch's
 * background pass has run (see apic_reconstruct).  Not thread-safe per plan.
 * Mixing with the device-pointer entries: apic_reconstruct, apic_reconstruct_u16, apic_reconstruct_prior,
 * apic_profile_begin (and apic_debug_copy for slot 0) use the same workspace as the pipeline slots, so each of them
 * first completes every batch that is still in flight, exactly as apic_wait_host would (the results are then in
 * the host buffers and a later apic_wait_host on that slot returns at once).  They never run beside a submitted
 * batch; a caller who wants overlap keeps to one family of entries per plan, or uses two plans. */
int apic_submit_host(apic_plan* plan, int slot, const float* h_intensity, int batch, float* h_field,
                     float* h_zernike, float* h_pupil, int32_t* h_status);
int apic_submit_host_u16(apic_plan* plan, int slot, const uint16_t* h_raw, const float* h_scale, int batch,
                         float* h_field, float* h_zernike, float* h_pupil, int32_t* h_status);
int apic_wait_host(apic_plan* plan, int slot);

/* Slide-level pupil prior (PAPER.md:171 / Fig. 4(b): the recovered pupil varies smoothly over
 * the slide; the use made of it is reading B9 of DESIGN.md).
 * apic_pupil_field_fit: d_zernike [tiles][n_zernike] (what apic_reconstruct returned), d_status [tiles], d_xy [tiles][2]
 * (slide coordinates of the tiles, any units; [-1, 1] keeps the fit well scaled) -> d_fit [tiles][n_zernike]: each
 * coefficient's least-squares polynomial of total degree `order` (0, 1, 2; terms 1, X, Y, X^2, XY, Y^2) over the tiles
 * with status 0, evaluated at EVERY tile; d_poly [6][n_zernike] the polynomial (unused terms 0).  If those tiles do not
 * determine the polynomial: their mean; none: zeros.  One small kernel on cuda_stream; device pointers; n_zernike <= 64.
 * apic_reconstruct_prior: apic_reconstruct whose aberration fit (S6) starts from d_zernike_init [batch][n_zernike]
 * (e.g. the rows of d_fit) instead of its own gradient-domain start; the re-wrapped refinement steps and the status
 * rule are unchanged, so a tile inside the basin of its own start gets the same coefficients, and a tile whose own
 * start lands in a wrong minimum (large aberrations on small tiles, R11) is rescued by its neighbours. */
int apic_pupil_field_fit(const float* d_zernike, const int32_t* d_status, const float* d_xy, int tiles, int n_zernike,
                         int order, float* d_fit, float* d_poly, void* cuda_stream);
int apic_reconstruct_prior(apic_plan* plan, const float* d_intensity, const float* d_zernike_init, int batch,
                           float* d_field, float* d_zernike, float* d_pupil, int32_t* d_status, void* cuda_stream);

/* Within-FOV reassembly of overlapping reconstructed tiles ("individually
 * reconstructed and then stitched together", "the overlapping regions were blended"; the blend and the
 * global-phase treatment are readings B6-B8 of DESIGN.md).  d_fields: [tiles_y][tiles_x][tile_px][tile_px] complex64
 * (the fields apic_reconstruct returns, tile_px = upsample * tile_n), tiles on a regular grid sharing `overlap` pixels
 * with each neighbour, 0 <= 2 overlap <= tile_px.  d_fov: [H][W] complex64, H = tiles_y (tile_px - overlap) + overlap
 * (W likewise): the separable linear blend of the tiles, each multiplied by its unit factor d_factors[tile] (complex64,
 * written by the call).  align != 0: the factors bring every tile to the global phase of tile (0, 0) in raster order
 * through the correlation of its overlaps with the left / upper neighbour (tiles come out of apic_reconstruct with
 * their own DC real-positive, so neighbours differ by a unit factor); align == 0: all factors 1.  d_work: device
 * scratch of apic_reassemble_work_bytes(tiles_y, tiles_x) bytes.  All pointers are DEVICE pointers owned by the caller;
 * the call only enqueues three kernels on cuda_stream.  Stateless (no plan).  Returns APIC_EINVAL on bad geometry. */
size_t apic_reassemble_work_bytes(int tiles_y, int tiles_x);
int apic_reassemble(const float* d_fields, int tiles_y, int tiles_x, int tile_px, int overlap, int align, float* d_fov,
                    float* d_factors, void* d_work, void* cuda_stream);

/* apic_reassemble for callers that cannot supply d_work because they cannot obtain device memory at the point
 * where they reassemble: a host program that gave all device memory to its own arena at start-up, a component
 * whose embedding application owns the allocator, a real-time acquisition loop in which a cudaMalloc / cudaFree
 * would stall every stream of the process.  Same arguments, same kernels and bit-identical results to
 * apic_reassemble, minus d_work: the scratch is a fixed array compiled into libapic's device image.
 *  - Limit: tiles_y * tiles_x <= apic_reassemble_static_max_tiles() (1024, e.g. a 32 x 32 FOV); beyond it the
 *    call returns APIC_ESCRATCH and enqueues nothing - use apic_reassemble with your own d_work then.  Every
 *    other argument is validated as in apic_reassemble (APIC_EINVAL).
 *  - Cost: the array (528 KiB) occupies memory on every GPU on which this library's device code gets loaded,
 *    from that moment until the process ends, used or not.
 *  - The call itself performs no cudaMalloc / cudaFree and calls no library routine that allocates; d_fields,
 *    d_fov and d_factors remain the caller's DEVICE buffers.
 *  - Set-up: the FIRST call on each device asks the CUDA runtime for the array's address on that device
 *    (cudaGetSymbolAddress, host-synchronous, may load the library's device code) and caches it; later calls
 *    on that device only enqueue the three kernels.  The device that owns the buffers must be current during
 *    every call.  Make that first call during initialisation, outside any stream capture.  A failed look-up
 *    returns APIC_ECUDA (text in apic_last_cuda_error) and is retried by the next call.
 *  - Sharing: all calls on one device, from any thread, stream or plan-less context, use the SAME array.  Calls
 *    whose kernels can overlap on the GPU (different streams without an ordering event between them) race on it
 *    and both results are undefined; order them on one stream or with events.  The array keeps whatever the last
 *    call wrote; no call depends on it (every element read is written earlier in the same call), so nothing is
 *    cleared between calls. */
int apic_reassemble_static_max_tiles(void);
int apic_reassemble_static(const float* d_fields, int tiles_y, int tiles_x, int tile_px, int overlap, int align,
                           float* d_fov, float* d_factors, void* cuda_stream);

/* Stage-level access for parity tests (device pointers, valid after apic_reconstruct on the
 * same stream, for the tiles of the LAST internal chunk; tile index is chunk-local):
 *   APIC_DBG_SUBSPECTRA: [chunk][sum_i |D_i|] complex64, S_hat_i on D_i (Eq. 7), LED-major, bins
 *                        of each disc in row-major order of the centred grid
 *   APIC_DBG_OBJECT_SPECTRUM: [chunk][N][N] complex64, O_hat in FFT order (bin k at index k mod N)
 *   APIC_DBG_DF_ITERS:   [chunk][n_dark_used] int32, CGLS iterations actually run
 */
enum { APIC_DBG_SUBSPECTRA = 0, APIC_DBG_OBJECT_SPECTRUM = 1, APIC_DBG_DF_ITERS = 2 };
int apic_debug_buffer(const apic_plan* plan, int which, void** d_ptr, size_t* bytes_per_tile);
/* Copies `tiles` tiles of that buffer into the caller's device buffer d_dst (asynchronously, on
 * cuda_stream). */
int apic_debug_copy(const apic_plan* plan, int which, void* d_dst, int tiles, void* cuda_stream);

/* Batched 2-D complex FFT used by every stage, exposed for kernel-level parity tests:
 * d_data [batch][n][n] complex64 transformed in place; forward = unnormalised e^{-j..}, inverse =
 * unnormalised e^{+j..}.  n in {64,128,256,512}. */
int apic_fft2d(float* d_data, int n, int batch, int inverse, void* cuda_stream);

/* The mixed-radix line transforms of the darkfield solver's reduced cyclic grids (lengths 16*R1,
 * R1 in {6,8,10,12,16}), exposed for kernel-level parity tests: d_data
 * [batch][my][mx] complex64 in place, mx, my in {96,128,160,192,256}.  mode 0 / 1: forward /
 * inverse 2-D DFT (unnormalised) by the "type X" transform; mode 2 / 3: per axis X inverse then
 * Y forward (2), or X forward then Y inverse (3), divided by the length: the identity. */
int apic_fft2d_xy(float* d_data, int mx, int my, int batch, int mode, void* cuda_stream);

/* Number of kernels launched by the last apic_reconstruct on this plan (bench's gpu_launches). */
int apic_last_launch_count(const apic_plan* plan);

/* Per-kernel timing for bench.py's roofline line.  Between apic_profile_begin and apic_profile_end
 * every `stride`-th launch of each kernel category made by apic_reconstruct on this plan is
 * bracketed by CUDA events on the launching stream (at most max_samples launches in total).
 * apic_profile_end synchronises those events and fills, per category (apic_profile_categories()
 * entries, named by apic_profile_category_name): the summed duration of the sampled launches in
 * ms, the number of sampled launches, and the number of all launches since apic_profile_begin. */
int apic_profile_categories(void);
const char* apic_profile_category_name(int cat);
int apic_profile_begin(apic_plan* plan, int stride, int max_samples);
int apic_profile_end(apic_plan* plan, double* ms_sum, long long* samples, long long* launches);
/* Nominal FFT flop (5 L log2 L per executed L-point line transform, counted by the kernels
 * themselves) of the darkfield kernels since apic_profile_begin (synchronises the device). */
int apic_profile_work(apic_plan* plan, unsigned long long* fft_flop);

/* Measured denominators for the roofline line (bench-side; not on the reconstruction path): runs a
 * register-resident loop on the current device, timed with CUDA events on cuda_stream, and returns
 * what = 0: fp32 FFMA rate in flop/s (2 per FMA); 1: fp32 FADD rate in flop/s (the FFT butterflies
 * are add-dominated); 2: shared-memory read bandwidth in bytes/s (conflict-free 16-byte loads). */
int apic_measure_peak(int what, double* per_second, void* cuda_stream);

const char* apic_strerror(int err);
const char* apic_last_cuda_error(void);
const char* apic_version(void);

#ifdef __cplusplus
}
#endif
#endif /* APIC_H_ */
