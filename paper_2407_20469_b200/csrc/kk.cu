// kk.cu - S0 image statistics / tile status and S1-S5 Kramers-Kronig field retrieval.
//
// S1-S5 (Eq. 4-7; readings R5-R7 in DESIGN.md): for each NA-matching image
//   l = log max(I, floor*mean I);  L = F(l);  G = w .* L (half-plane weights of Eq. 5);
//   s = exp(F^-1 G);  S_hat = F(s)/N^2 kept on the disc D_i only.
// Four strip kernels per image, every 1-D transform done in shared memory (fft_core.cuh):
//   kk_log_rowfft : log + row FFT              [y][x]  -> [y][kx]
//   kk_col_mask   : column FFT, w, column IFFT [y][kx] -> [ky][kx] -> [y][kx]
//   kk_row_exp    : row IFFT, exp, row FFT     [y][kx] -> [y][x]   -> [y][kx]
//   kk_col_gather : column FFT on the disc's columns only, gather D_i
#include <algorithm>

#include "fft_core.cuh"
#include "plan.hpp"

namespace apic {

// ---------------------------------------------------------------------------------- S0 statistics
// one CTA per (image, tile): sum, sum of squares and non-finite count of the image.  Thread i takes pixels
// 4 i .. 4 i + 3 (+ 1024 k) in both input forms, with the same association, so that the statistics of the
// uint16 entry equal those of the fp32 entry on float(count) * scale bit for bit.
template <bool U16>
__global__ void __launch_bounds__(256) image_stats_kernel(ImgSrc src, int npix, int n_img, double* __restrict__ stats) {
  const int img = blockIdx.x, tile = blockIdx.y;
  const size_t ii = size_t(tile) * n_img + img;
  float s = 0.f, q = 0.f;
  int bad = 0;
  if (U16) {
    const uint2* p = reinterpret_cast<const uint2*>(src.u16 + ii * npix);      // 4 pixels
    const float sc = src.scale[ii];
    for (int i = threadIdx.x; i < npix / 4; i += 256) {
      const uint2 r = __ldg(&p[i]);
      float4 v;
      v.x = float(r.x & 0xffffu) * sc; v.y = float(r.x >> 16) * sc; v.z = float(r.y & 0xffffu) * sc; v.w = float(r.y >> 16) * sc;
      s += (v.x + v.y) + (v.z + v.w);
      q += (v.x * v.x + v.y * v.y) + (v.z * v.z + v.w * v.w);
    }
    bad = (!isfinite(sc) && threadIdx.x == 0) ? 1 : 0;                         // counts are finite; a non-finite scale is bad input
  } else {
    const float4* p = reinterpret_cast<const float4*>(src.f32 + ii * npix);
    for (int i = threadIdx.x; i < npix / 4; i += 256) {
      float4 v = __ldg(&p[i]);
      bad += !isfinite(v.x) + !isfinite(v.y) + !isfinite(v.z) + !isfinite(v.w);
      s += (v.x + v.y) + (v.z + v.w);
      q += (v.x * v.x + v.y * v.y) + (v.z * v.z + v.w * v.w);
    }
  }
  __shared__ double sh[3][256];
  sh[0][threadIdx.x] = s;
  sh[1][threadIdx.x] = q;
  sh[2][threadIdx.x] = bad;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sh[0][threadIdx.x] += sh[0][threadIdx.x + o];
      sh[1][threadIdx.x] += sh[1][threadIdx.x + o];
      sh[2][threadIdx.x] += sh[2][threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x < 3) stats[ii * 3 + threadIdx.x] = sh[threadIdx.x][0];
}

void launch_image_stats(const DevTables& t, const ImgSrc& src, int batch, double* stats, const LaunchCtx& c) {
  dim3 grid(t.n_img, batch);
  ProfScope ps(c, CAT_STATS);
  if (src.u16) image_stats_kernel<true><<<grid, 256, 0, c.stream>>>(src, t.n * t.n, t.n_img, stats);
  else image_stats_kernel<false><<<grid, 256, 0, c.stream>>>(src, t.n * t.n, t.n_img, stats);
}

// one warp: per-tile status (O1, BASELINE.json item 5, R18) and the ordered list of
// tiles to reconstruct
__global__ void tile_status_kernel(const double* __restrict__ stats, int batch, int n_img, int nb, int npix,
                                   int bg_mode, float bg_thr, int32_t* __restrict__ status,
                                   int32_t* __restrict__ live, int32_t* __restrict__ live_count) {
  const int lane = threadIdx.x;
  int count = 0;
  for (int base = 0; base < batch; base += 32) {
    const int tile = base + lane;
    int st = -1;
    if (tile < batch) {
      const double* p = stats + size_t(tile) * n_img * 3;
      double bad = 0, sum = 0, sq = 0;
      for (int i = 0; i < n_img; ++i) bad += p[3 * i + 2];
      for (int i = 0; i < nb; ++i) { sum += p[3 * i]; sq += p[3 * i + 1]; }
      const double cnt = double(nb) * npix;
      const double mean = sum / cnt;
      st = 0;
      if (bad > 0) st = 2;
      else if (bg_mode == 1 && mean >= double(bg_thr)) st = 1;
      else if (bg_mode == 2 && (sq / cnt - mean * mean) / (mean * mean) <= double(bg_thr)) st = 1;
      status[tile] = st;
    }
    const unsigned m = __ballot_sync(0xffffffffu, st == 0);
    if (st == 0) live[count + __popc(m & ((1u << lane) - 1u))] = tile;
    count += __popc(m);
  }
  if (lane == 0) *live_count = count;
}

void launch_tile_status(const DevTables& t, const double* stats, int batch, int bg_mode, float bg_thr,
                        int32_t* status, int32_t* live, int32_t* live_count, const LaunchCtx& c) {
  ProfScope ps(c, CAT_STATS);
  tile_status_kernel<<<1, 32, 0, c.stream>>>(stats, batch, t.n_img, t.nb, t.n * t.n, bg_mode, bg_thr, status, live,
                                             live_count);
}

// background / bad-input tiles: outputs are zero
__global__ void __launch_bounds__(256) zero_dead_kernel(const int32_t* __restrict__ status, size_t field_f4,
                                                        int nz, size_t pupil_f4, float4* __restrict__ field,
                                                        float* __restrict__ zern, float4* __restrict__ pupil) {
  const int tile = blockIdx.y;
  const int st = status[tile];
  if (st != 1 && st != 2) return;
  const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
  const size_t stride = size_t(gridDim.x) * 256, t0 = size_t(blockIdx.x) * 256 + threadIdx.x;
  for (size_t i = t0; i < field_f4; i += stride) field[size_t(tile) * field_f4 + i] = z;
  if (pupil)
    for (size_t i = t0; i < pupil_f4; i += stride) pupil[size_t(tile) * pupil_f4 + i] = z;
  if (blockIdx.x == 0 && threadIdx.x < nz) zern[size_t(tile) * nz + threadIdx.x] = 0.f;
}

void launch_zero_dead(const DevTables& t, const int32_t* status, int batch, float* field, float* zern,
                      float* pupil, const LaunchCtx& c) {
  const size_t on = size_t(t.n) * t.u;
  dim3 grid(32, batch);
  ProfScope ps(c, CAT_STATS);
  zero_dead_kernel<<<grid, 256, 0, c.stream>>>(status, on * on * 2 / 4, t.nz, size_t(t.n) * t.n * 2 / 4,
                                               reinterpret_cast<float4*>(field), zern,
                                               reinterpret_cast<float4*>(pupil));
}

// ---------------------------------------------------------------------------------- S1-S2
// PADDED (kk_pad 2, R7): the image, Fourier-interpolated to the N = 2 x tile_n grid, is already in G (kk_pad_* below);
// its real part is the input and the row is transformed in place.
template <int N, bool PADDED>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB)
kk_log_rowfft(DevTables t, ImgSrc src, const double* __restrict__ stats, float floor_rel,
              float2* __restrict__ G, const int32_t* __restrict__ live, const int32_t* __restrict__ live_count,
              int chunk0) {
  using S = Strip<N>;
  using TH = StripThread<N, false>;
  extern __shared__ float2 sm[];
  const int slot = blockIdx.z, led = blockIdx.y;
  const int tile = resolve_tile_idx(live, live_count, chunk0, slot);
  if (tile < 0) return;
  const int line = TH::line(), tt = TH::t(), y = blockIdx.x * S::LINES + line;
  const size_t ii = size_t(tile) * t.n_img + led;
  const float mean = float(stats[(size_t(tile) * t.n_img + led) * 3] / double(t.n * t.n));   // interpolation keeps the mean
  const float lo = floor_rel * mean;                                   // R6
  float2* g = G + (size_t(slot) * t.nb + led) * (N * N) + y * N;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const float x = PADDED ? g[tt + S::TPL * r].x : img_load(src, ii, N * N, y * N + tt + S::TPL * r);
    v[r] = make_float2(logf(fmaxf(x, lo)), 0.f);                        // Re of Eq. 4
  }
  fft_regs<N, false>(v, sm + line * S::LS, tt, t.tw_kk);
#pragma unroll
  for (int r = 0; r < S::R; ++r) g[tt + S::TPL * r] = v[r];
}

// ---------------------------------------------------------------------------------- S2-S4
template <int N>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB)
kk_col_mask(DevTables t, float2* __restrict__ G, const int32_t* __restrict__ live_count, int chunk0) {
  using S = Strip<N>;
  using TH = StripThread<N, true>;
  extern __shared__ float2 sm[];
  const int slot = blockIdx.z, led = blockIdx.y;
  if (chunk0 + slot >= *live_count) return;
  const int line = TH::line(), tt = TH::t(), x = blockIdx.x * S::LINES + line;
  float2* g = G + (size_t(slot) * t.nb + led) * (N * N) + x;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) v[r] = g[(tt + S::TPL * r) * N];
  fft_regs<N, false>(v, sm + line * S::LS, tt, t.tw_kk);
  const uint8_t* w2 = t.halfplane2 + size_t(led) * (N * N) + x;
  const float scale = 0.5f / float(N * N);                              // w = w2/2, and the 1/N^2 of F^-1
#pragma unroll
  for (int r = 0; r < S::R; ++r) v[r] = cscale(v[r], float(__ldg(&w2[(tt + S::TPL * r) * N])) * scale);   // Eq. 5
  fft_regs<N, true>(v, sm + line * S::LS, tt, t.tw_kk);
#pragma unroll
  for (int r = 0; r < S::R; ++r) g[(tt + S::TPL * r) * N] = v[r];
}

// ---------------------------------------------------------------------------------- S4-S5
template <int N>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB)
kk_row_exp(DevTables t, float2* __restrict__ G, const int32_t* __restrict__ live_count, int chunk0) {
  using S = Strip<N>;
  using TH = StripThread<N, false>;
  extern __shared__ float2 sm[];
  const int slot = blockIdx.z, led = blockIdx.y;
  if (chunk0 + slot >= *live_count) return;
  const int line = TH::line(), tt = TH::t(), y = blockIdx.x * S::LINES + line;
  float2* g = G + (size_t(slot) * t.nb + led) * (N * N) + y * N;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) v[r] = g[tt + S::TPL * r];
  fft_regs<N, true>(v, sm + line * S::LS, tt, t.tw_kk);
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const float a = expf(v[r].x);                                       // Eq. 6
    float sn, cs;
    sincosf(v[r].y, &sn, &cs);
    v[r] = make_float2(a * cs, a * sn);
  }
  fft_regs<N, false>(v, sm + line * S::LS, tt, t.tw_kk);
#pragma unroll
  for (int r = 0; r < S::R; ++r) g[tt + S::TPL * r] = v[r];
}

// ---------------------------------------------------------------------------------- S5 (Eq. 7)
template <int N>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB)
kk_col_gather(DevTables t, const float2* __restrict__ G, float2* __restrict__ Sp,
              const int32_t* __restrict__ live_count, int chunk0) {
  using S = Strip<N>;
  using TH = StripThread<N, true>;
  extern __shared__ float2 sm[];
  const int slot = blockIdx.z, led = blockIdx.y, c0 = blockIdx.x * S::LINES;
  if (chunk0 + slot >= *live_count) return;
  const int ncol = t.bf_ncol[led];
  if (c0 >= ncol) return;
  const int line = TH::line(), tt = TH::t(), c = c0 + line;
  const bool valid = c < ncol;
  const int fx = (t.bf_col0[led] + c + N) & (N - 1);
  const float2* g = G + (size_t(slot) * t.nb + led) * (N * N) + fx;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) v[r] = valid ? g[(tt + S::TPL * r) * N] : make_float2(0.f, 0.f);
  fft_regs<N, false>(v, sm + line * S::LS, tt, t.tw_kk);
  if (!valid) return;
  const int32_t* map = t.bf_map + t.bf_map_off[led] + c;
  float2* s = Sp + size_t(slot) * t.disc_total;
  const float scale = 1.f / float(N * N);
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int ent = __ldg(&map[(tt + S::TPL * r) * ncol]);
    if (ent >= 0) s[ent] = cscale(v[r], scale);
  }
}

// ---------------------------------------------------------------------------------- kk_pad 2 (R7)
// image -> complex N x N grid (the input of the N-grid transform)
__global__ void __launch_bounds__(256) kk_pad_load(DevTables t, ImgSrc src, float2* __restrict__ KP,
                                                   const int32_t* __restrict__ live, const int32_t* __restrict__ live_count,
                                                   int chunk0) {
  const int slot = blockIdx.z, led = blockIdx.y;
  const int tile = resolve_tile_idx(live, live_count, chunk0, slot);
  if (tile < 0) return;
  const int nn = t.n * t.n;
  const size_t ii = size_t(tile) * t.n_img + led;
  float2* k = KP + (size_t(slot) * t.nb + led) * nn;
  for (int q = blockIdx.x * 256 + threadIdx.x; q < nn; q += gridDim.x * 256) k[q] = make_float2(img_load(src, ii, nn, q), 0.f);
}
// spectrum on the N grid -> zero-padded spectrum on the M = 2N grid, / N^2, the sign-less Nyquist row and column of
// the N grid split evenly between +N/2 and -N/2 (band-limited interpolation: values at the common points are kept)
__global__ void __launch_bounds__(256) kk_pad_scatter(DevTables t, const float2* __restrict__ KP, float2* __restrict__ G,
                                                      const int32_t* __restrict__ live_count, int chunk0) {
  const int slot = blockIdx.z, led = blockIdx.y;
  if (chunk0 + slot >= *live_count) return;
  const int n = t.n, m = t.kk_n, h = n / 2;
  const float2* k = KP + (size_t(slot) * t.nb + led) * (n * n);
  float2* g = G + (size_t(slot) * t.nb + led) * (size_t(m) * m);
  const float inv = 1.f / float(n * n);
  for (int q = blockIdx.x * 256 + threadIdx.x; q < m * m; q += gridDim.x * 256) {
    const int fy = q / m, fx = q - fy * m;
    const int ky = fy < m / 2 ? fy : fy - m, kx = fx < m / 2 ? fx : fx - m;     // signed bins of the M grid
    float w = inv;
    if (ky < -h || ky > h || kx < -h || kx > h) w = 0.f;
    if (ky == -h || ky == h) w *= 0.5f;
    if (kx == -h || kx == h) w *= 0.5f;
    float2 v = make_float2(0.f, 0.f);
    if (w != 0.f) v = cscale(k[((ky + n) & (n - 1)) * n + ((kx + n) & (n - 1))], w);
    g[q] = v;
  }
}

template <int N, bool PADDED>
static void launch_kk_n(const DevTables& t, const Workspace& w, const LaunchCtx& c, const ImgSrc& src,
                        const double* stats, float floor_rel) {
  using S = Strip<N>;
  constexpr int TH = S::THREADS;
  constexpr size_t SM = S::SMEM;
  if (!c.pd->attr_kk) {
    cudaFuncSetAttribute(kk_log_rowfft<N, PADDED>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
    cudaFuncSetAttribute(kk_col_mask<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
    cudaFuncSetAttribute(kk_row_exp<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
    cudaFuncSetAttribute(kk_col_gather<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
    c.pd->attr_kk = true;
  }
  if (PADDED) {
    // I -> F_N(I) -> zero-padded to the 2N grid -> F_2N^-1: the interpolated image (its real part is used)
    ProfScope ps(c, CAT_KK_LOG_ROWFFT);
    const int images = c.chunk_tiles * t.nb;
    kk_pad_load<<<dim3(16, t.nb, c.chunk_tiles), 256, 0, c.stream>>>(t, src, w.KP, c.live, c.live_count, c.chunk0);
    launch_fft2d(w.KP, t.n, images, false, t.tw, c.stream);
    kk_pad_scatter<<<dim3(64, t.nb, c.chunk_tiles), 256, 0, c.stream>>>(t, w.KP, w.G, c.live_count, c.chunk0);
    launch_fft2d(w.G, N, images, true, t.tw_kk, c.stream);
    *c.launches += 5;                       // load, 2 + 2 transform passes, scatter (the scope above counted one)
  }
  // The four strip kernels alternate between row and column strips, so every kernel boundary is a transposition
  // through memory.  The grids of a whole pass (nb N^2 complex64 per tile: 268 MB for 64 tiles of config 2) do not fit
  // the L2, so the pass is cut into sub-passes whose grids do (two sub-passes in flight on two streams, so that the
  // launch tails of one overlap the other): only the images in and the sub-spectra out touch HBM.
  const size_t per_tile = size_t(t.nb) * N * N * sizeof(float2);
  int sub = c.chunk_tiles;
  if (!PADDED && c.aux && per_tile * c.chunk_tiles > size_t(c.pd->l2_bytes) * 4 / 10) {
    sub = std::max(1, int(size_t(c.pd->l2_bytes) * 4 / 10 / per_tile));
    const int n_sub = (c.chunk_tiles + sub - 1) / sub;
    sub = (c.chunk_tiles + n_sub - 1) / n_sub;            // balanced
  }
  const bool split = sub < c.chunk_tiles;
  if (split) {
    cudaEventRecord(c.ev_fork, c.stream);
    cudaStreamWaitEvent(c.aux, c.ev_fork, 0);
  }
  int k = 0;
  for (int s0 = 0; s0 < c.chunk_tiles; s0 += sub, ++k) {
    const int ns = std::min(sub, c.chunk_tiles - s0);
    LaunchCtx cs = c;
    cs.stream = (split && (k & 1)) ? c.aux : c.stream;
    // a sub-pass reuses the grid region of the sub-pass two before it (same stream, so ordered): the dead grids are
    // overwritten while they still sit in L2 instead of being written back to HBM
    float2* G = w.G + size_t(split ? (k & 1) * sub : s0) * t.nb * N * N;
    float2* Sp = w.S + size_t(s0) * t.disc_total;
    const int ch0 = c.chunk0 + s0;
    dim3 grid(N / S::LINES, t.nb, ns);
    { ProfScope ps(cs, CAT_KK_LOG_ROWFFT);
      kk_log_rowfft<N, PADDED><<<grid, TH, SM, cs.stream>>>(t, src, stats, floor_rel, G, c.live, c.live_count, ch0); }
    { ProfScope ps(cs, CAT_KK_COL_MASK);
      kk_col_mask<N><<<grid, TH, SM, cs.stream>>>(t, G, c.live_count, ch0); }
    { ProfScope ps(cs, CAT_KK_ROW_EXP);
      kk_row_exp<N><<<grid, TH, SM, cs.stream>>>(t, G, c.live_count, ch0); }
    dim3 grid4((t.bf_max_ncol + S::LINES - 1) / S::LINES, t.nb, ns);
    { ProfScope ps(cs, CAT_KK_COL_GATHER);
      kk_col_gather<N><<<grid4, TH, SM, cs.stream>>>(t, G, Sp, c.live_count, ch0); }
  }
  if (split) {
    cudaEventRecord(c.ev_join, c.aux);
    cudaStreamWaitEvent(c.stream, c.ev_join, 0);
  }
}

void launch_kk(const DevTables& t, const Workspace& w, const LaunchCtx& c, const ImgSrc& src, const double* stats,
               float floor_rel) {
  if (t.kk_n == t.n) {
    switch (t.n) {
      case 64: launch_kk_n<64, false>(t, w, c, src, stats, floor_rel); break;
      case 128: launch_kk_n<128, false>(t, w, c, src, stats, floor_rel); break;
      case 256: launch_kk_n<256, false>(t, w, c, src, stats, floor_rel); break;
      case 512: launch_kk_n<512, false>(t, w, c, src, stats, floor_rel); break;
    }
  } else {                                   // kk_pad 2: the chain runs on the 2N grid
    switch (t.kk_n) {
      case 128: launch_kk_n<128, true>(t, w, c, src, stats, floor_rel); break;
      case 256: launch_kk_n<256, true>(t, w, c, src, stats, floor_rel); break;
      case 512: launch_kk_n<512, true>(t, w, c, src, stats, floor_rel); break;
    }
  }
}

// ---------------------------------------------------------------------------------- plain 2-D FFT
template <int N, bool INV, bool COLS>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB)
fft_pass_kernel(float2* __restrict__ d, const float2* __restrict__ tw) {
  using S = Strip<N>;
  using TH = StripThread<N, COLS>;
  extern __shared__ float2 sm[];
  const int line = TH::line(), tt = TH::t(), l = blockIdx.x * S::LINES + line;
  float2* g = d + size_t(blockIdx.y) * (N * N) + (COLS ? l : l * N);
  constexpr int STR = COLS ? N : 1;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) v[r] = g[(tt + S::TPL * r) * STR];
  fft_regs<N, INV>(v, sm + line * S::LS, tt, tw);
#pragma unroll
  for (int r = 0; r < S::R; ++r) g[(tt + S::TPL * r) * STR] = v[r];
}

template <int N>
static int fft2d_n(float2* d, int batch, bool inverse, const float2* tw, cudaStream_t s) {
  using S = Strip<N>;
  constexpr int TH = S::THREADS;
  constexpr size_t SM = S::SMEM;
  cudaFuncSetAttribute(fft_pass_kernel<N, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
  cudaFuncSetAttribute(fft_pass_kernel<N, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
  cudaFuncSetAttribute(fft_pass_kernel<N, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
  cudaFuncSetAttribute(fft_pass_kernel<N, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
  for (int b0 = 0; b0 < batch; b0 += 32768) {
    const int nb = batch - b0 < 32768 ? batch - b0 : 32768;
    dim3 grid(N / S::LINES, nb);
    float2* p = d + size_t(b0) * (N * N);
    if (inverse) {
      fft_pass_kernel<N, true, false><<<grid, TH, SM, s>>>(p, tw);
      fft_pass_kernel<N, true, true><<<grid, TH, SM, s>>>(p, tw);
    } else {
      fft_pass_kernel<N, false, false><<<grid, TH, SM, s>>>(p, tw);
      fft_pass_kernel<N, false, true><<<grid, TH, SM, s>>>(p, tw);
    }
  }
  return 0;
}

int launch_fft2d(float2* d, int n, int batch, bool inverse, const float2* tw, cudaStream_t s) {
  switch (n) {
    case 64: return fft2d_n<64>(d, batch, inverse, tw, s);
    case 128: return fft2d_n<128>(d, batch, inverse, tw, s);
    case 256: return fft2d_n<256>(d, batch, inverse, tw, s);
    case 512: return fft2d_n<512>(d, batch, inverse, tw, s);
  }
  return -1;
}

}  // namespace apic
