// plan.hpp - device-side view of an apic_plan: geometry tables (read-only, identical for every
// tile) and the per-chunk workspace.  Shared by the kernel translation units and api.cu.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <vector>

#include "geometry.hpp"

namespace apic {

struct DevTables {
  int n, u, nb, nd, nz, n_img;   // n_img = nb + nd
  const float2* tw;              // twiddle tables of fft_core.cuh (build_twiddles)
  int kk_n;                      // grid of the KK step, kk_pad * N (R7)
  const float2* tw_kk;           // twiddles of the kk_n-point line transform (= tw when kk_pad = 1)
  const float2* tw_xy;           // [5][256] twiddles of fft_xy.cuh for R1 = 6, 8, 10, 12, 16 (N = 256 only)
  // NA-matching side
  const uint8_t* halfplane2;     // [nb][kk_n*kk_n] FFT order, 2*w of Eq. 5
  int disc_total;                // sum_i |D_i|
  const float* disc_zern;        // [disc_total][nz]  Z_j(K+kappa_i) - Z_j(kappa_i)
  const int32_t* bf_col0;        // [nb]
  const int32_t* bf_ncol;        // [nb]
  const int32_t* bf_map_off;     // [nb+1]
  const int32_t* bf_map;         // per LED [kk_n(fy)][ncol] -> flattened entry | -1
  int bf_max_ncol;
  // aberration system
  int n_rows, n_grad;
  const int32_t* row_src;        // [n_rows][2]
  const float* a_full;           // [nz][n_rows] (transposed on upload)
  const int32_t* grad_rows;      // [n_grad][2]
  // stitching
  int n_union;
  const int32_t* union_f;        // [n_union]
  const int32_t* union_off;      // [n_union+1]
  const int32_t* union_src;
  // output
  int known_row0, known_nrow;    // centred ky range of the final known region
  const float2* ramp;            // [u][N]: e^{+2 pi i k a / (uN)}, index a*N + (k mod N), k signed bin
  int n_pupil;
  const int32_t* pupil_idx;      // centred linear index
  const float* pupil_zern;       // [n_pupil][nz]
};


struct DarkDev {
  int n_unknown, n_disc, n_eq;
  int d_col0, d_ncol, d_row0, d_nrow;   // disc bbox (centred)
  int u_row0, u_nrow;                   // rows holding unknown bins
  int q_col0, q_ncol, q_row0, q_nrow;   // bbox of the linear region Q
  const int32_t* disc_f;                // [n_disc] FFT-order index (U entries first)
  const float* zern;                    // [n_disc][nz] Z_j(K + kappa)
  const int32_t* dmap;                  // [N(fy)][d_ncol] -> disc entry | -1
  const int32_t* qmap;                  // [N(fy)][q_ncol] -> equation | -1
  int led;                              // input index among the darkfield LEDs
  int mx, my;                           // reduced cyclic grid of the CG mat-vecs (geometry.hpp)
  const int32_t* dmap_m;                // [my][mx] -> disc entry | -1
  const uint8_t* qmask_m;               // [my][mx] -> 1 on Q
  int u_strip_off[kMaxUStrips + 1];     // first U entry of each 16-row strip of the U rows (U entries are row-major)
  int u0m, q0m, d0m;                    // u_row0, q_row0, d_row0 mod my (first physical row on the reduced grid)
  int accumulate;                       // df_order 1: the extension step adds to O instead of assigning
  int n_avg;                            // last LED of a ring (df_order 1): bins solved by c >= 2 LEDs of the ring ...
  const int32_t* avg_f;                 // ... their FFT-order index
  const float* avg_w;                   // ... and 1 / c
};

constexpr int kGramRows = 512;          // rows per Gram partial (aberration kernels)
constexpr int kMaxZern = 64;

struct Workspace {
  int chunk;               // tiles per pass
  float2* G;               // [chunk][nb][kk_n*kk_n] KK working grids
  float2* KP;              // [chunk][nb][N*N]   spectra of the intensities on the N grid (kk_pad 2 only)
  float2* S;               // [chunk][disc_total] sub-spectra on the discs (Eq. 7)
  float2* PR;              // [chunk][n_rows]    p = S_i conj S_l on the overlaps (Eq. 9)
  float* gram;             // [chunk][gram_parts][gram_entries]
  int gram_parts, gram_entries;
  float* coef;             // [chunk][nz]
  int32_t* ab_fail;        // [chunk] Cholesky failure flag
  float2* O;               // [chunk][N*N] object spectrum, FFT order
  float2* T;               // [chunk][N*N] transform scratch
  float2* PF;              // [chunk][N*N] p = F^-1 P_hat of the current darkfield LED
  float2* TM;              // [chunk][N*N] transform scratch on the reduced grid (df_mgrid.cu)
  float2* vec_w;           // [chunk][max_unknown] w = C^H M_Q C pdir of the current CG iteration
  float2* vec_x;           // [chunk][max_unknown] CG iterate
  float2* vec_s;           // [chunk][max_unknown] CG residual of the normal equations
  int32_t* cg_iters;       // [chunk][n_dark_used]
  unsigned long long* df_work;   // [1] nominal flop (5 L log2 L per L-point line transform) executed by the darkfield kernels
  float2* TOUT;            // [chunk][N][uN]
  int max_eq, max_unknown;
};

// Where a step's intensities come from: fp32 values in radiometric units (apic_reconstruct) or raw uint16
// camera counts with one factor per image (apic_reconstruct_u16; PAPER.md:199 - exposures differ between
// NA-matching and darkfield frames).  The conversion count * scale happens in the load itself, in fp32, so both
// entries see the same bits for the same values and no fp32 working copy of the counts exists.
struct ImgSrc {
  const float* f32;        // [batch][n_img][N*N] or nullptr
  const uint16_t* u16;     // [batch][n_img][N*N] or nullptr
  const float* scale;      // [batch][n_img] (uint16 form only)
};

// Batch-level state
struct BatchState {
  double* stats;           // [max_batch][n_img][3]: sum, sum of squares, non-finite count
  int32_t* live;           // [max_batch] compacted list of tiles to reconstruct
  int32_t* live_count;     // device scalar
};

// ------------------------------------------------------------------ per-kernel timing (apic_profile_*)
enum KernelCat {
  CAT_STATS = 0, CAT_KK_LOG_ROWFFT, CAT_KK_COL_MASK, CAT_KK_ROW_EXP, CAT_KK_COL_GATHER, CAT_AB_PRODUCTS, CAT_AB_GRAM,
  CAT_AB_SOLVE, CAT_STITCH, CAT_OUT_ROWS, CAT_OUT_COLS, CAT_PUPIL, CAT_DF_MGRID, CAT_DF_TEAM, CAT_DF_TMA, CAT_DF_WIDE, CAT_COUNT
};

// Per-plan record of what has been set up on the plan's device (function attributes are per device, so the
// flags live in the plan, not in process-wide statics: a second plan on another GPU does its own set-up).
struct PlanDevice {
  int device = 0;          // CUDA device the plan was created on (apic_reconstruct runs there)
  int sms = 0;             // its SM count
  int l2_bytes = 0;        // its L2 size
  bool attr_kk = false, attr_ab = false, attr_out = false, attr_team = false, attr_mgrid = false, attr_tma = false;
};

struct Profiler {
  bool on = false;
  int stride = 1;
  std::vector<cudaEvent_t> ev;     // pool of (start, end) pairs
  std::vector<int> cat;            // category of each used pair
  int used = 0;
  long long launches[CAT_COUNT] = {0};
};

// ------------------------------------------------------------------ launchers (one per kernel)
struct LaunchCtx {
  cudaStream_t stream;
  int* launches;           // counter
  Profiler* prof;
  const int32_t* live;     // compacted tile list
  const int32_t* live_count;
  int chunk0;              // first live-list position of this chunk
  int chunk_tiles;         // grid size in tiles (CTAs beyond live_count exit)
  PlanDevice* pd;          // per-plan device state (attribute set-up flags, SM count)
  cudaStream_t aux = nullptr;          // second stream of this workspace set (KK sub-passes alternate between the two) ...
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;   // ... and the events that fork it from / join it into `stream`
};

// stats / status (batch-level)
// Brackets one kernel launch: counts it and, when profiling samples it, records CUDA events around it.
struct ProfScope {
  Profiler* p;
  cudaStream_t s;
  int slot = -1;
  ProfScope(const LaunchCtx& c, int cat) : p(c.prof), s(c.stream) {
    ++*c.launches;
    if (!p) return;
    const long long k = p->launches[cat]++;
    if (!p->on || k % p->stride != 0 || size_t(2 * p->used + 2) > p->ev.size()) return;
    slot = p->used++;
    p->cat[slot] = cat;
    cudaEventRecord(p->ev[2 * slot], s);
  }
  ~ProfScope() {
    if (slot >= 0) cudaEventRecord(p->ev[2 * slot + 1], s);
  }
};

void launch_image_stats(const DevTables& t, const ImgSrc& src, int batch, double* stats, const LaunchCtx& c);
void launch_tile_status(const DevTables& t, const double* stats, int batch, int bg_mode, float bg_thr,
                        int32_t* status, int32_t* live, int32_t* live_count, const LaunchCtx& c);
void launch_zero_dead(const DevTables& t, const int32_t* status, int batch, float* field, float* zern,
                      float* pupil, const LaunchCtx& c);

// KK (S1-S5)
void launch_kk(const DevTables& t, const Workspace& w, const LaunchCtx& c, const ImgSrc& src,
               const double* stats, float floor_rel);
// aberration (S6) + stitching (S7)
// d_init != nullptr: [batch][nz] prior coefficients (indexed by tile) that replace the gradient-domain start (reading B9)
void launch_aberration(const DevTables& t, const Workspace& w, const LaunchCtx& c, int refine_iters,
                       float* d_zernike, int32_t* d_status, const float* d_init = nullptr);
void launch_stitch(const DevTables& t, const Workspace& w, const LaunchCtx& c);
// darkfield (S8-S10), every LED in one launch (df_team.cu)
void launch_darkfield_team(const DevTables& t, const DarkDev* d_leds, int n_leds, const Workspace& w, const LaunchCtx& c,
                           const ImgSrc& src, int df_iters, float df_tol, int team_size);
// darkfield (S8-S10) on reduced cyclic grids, every LED in one launch (df_mgrid.cu; N = 256)
void launch_darkfield_mgrid(const DevTables& t, const DarkDev* d_leds, int n_leds, const Workspace& w, const LaunchCtx& c,
                            const ImgSrc& src, int df_iters, float df_tol, int team_size);
// the same solver with strips staged by the async proxy (cp.async.bulk + mbarrier) and distributed CG vectors
// (df_tma.cu; N = 256, df_mode 4); h_leds = host copy of d_leds
void launch_darkfield_tma(const DevTables& t, const DarkDev* d_leds, const DarkDev* h_leds, int n_leds, const Workspace& w,
                          const LaunchCtx& c, const ImgSrc& src, int df_iters, float df_tol, int team_size);
// the same solver scheduled wide: NG strip groups of 256 threads per CTA at 64 registers, p_M strips parked in shared
// memory, distributed CG vectors (df_wide.cu; N = 256, df_mode 5).  false: the configuration does not fit.
bool launch_darkfield_wide(const DevTables& t, const DarkDev* d_leds, const DarkDev* h_leds, int n_leds, const Workspace& w,
                           const LaunchCtx& c, const ImgSrc& src, int df_iters, float df_tol, int team_size, int groups);
int launch_fft2d_xy(float2* d, int mx, int my, int batch, int mode, const float2* tw_xy, cudaStream_t s);
// outputs
void launch_output(const DevTables& t, const Workspace& w, const LaunchCtx& c, float* d_field, float* d_pupil);

// plain batched 2-D FFT (apic_fft2d)
int launch_fft2d(float2* d, int n, int batch, bool inverse, const float2* tw, cudaStream_t s);

#ifdef __CUDACC__
// pixel `px` of image `img` (= tile * n_img + led) of `npix` pixels, in radiometric units
__device__ __forceinline__ float img_load(const ImgSrc& s, size_t img, int npix, int px) {
  if (s.u16) return float(__ldg(&s.u16[img * size_t(npix) + px])) * __ldg(&s.scale[img]);
  return __ldg(&s.f32[img * size_t(npix) + px]);
}
// tile handled by chunk-local slot `slot` (-1: beyond the live list)
__device__ __forceinline__ int resolve_tile_idx(const int32_t* __restrict__ live,
                                                const int32_t* __restrict__ live_count, int chunk0, int slot) {
  const int pos = chunk0 + slot;
  if (pos >= *live_count) return -1;
  return live[pos];
}
#endif

}  // namespace apic
