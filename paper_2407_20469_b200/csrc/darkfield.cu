// darkfield.cu - S8-S10 darkfield extension (Eq. 11-13; readings R15-R17).
//
// For one darkfield LED (processing order = ascending |kappa|):
//   P_hat = O_hat e^{j phi(k+kappa)} on P = D_i ∩ known,   p = F^-1 P_hat,
//   d     = [F(I_i)/N^2 - P_hat ⋆ P_hat] on Q = F(I_i - |p|^2)/N^2 on Q          (Eq. 13 lhs)
//   (C u)(k)   = (1/N^2) F[conj(p) . F^-1(E_U u)](k), k in Q                     (block-Toeplitz C,
//   (C^H v)(u) = (1/N^2) F[p . F^-1(M_Q v)](u),        u in U                     PAPER.md:135)
//   U_hat = argmin ||C u - d||  by conjugate gradients on the normal equations, never forming C
//   (the paper builds C explicitly: ~90 % of its run time),
//   O_hat(u) = U_hat(u) e^{-j phi(u+kappa)}, known ∪= U.
// Transforms are pruned to the rows that hold data: U/P rows (~2R+1) and Q rows (<= 4R+1).
// One CG iteration = 5 strip kernels + one vector update:
//   A rows_u_scatter (E_U pdir, row IFFT) -> B cols_mul<conj> (col IFFT, .conj p, col FFT)
//   -> C rows_q (row FFT, mask Q / N^2, row IFFT) -> D cols_mul (col IFFT, .p, col FFT)
//   -> E rows_u_gather (row FFT, gather U: w = C^H C pdir, partial <pdir,w>) -> F cg_update.
#include "fft_core.cuh"
#include "plan.hpp"

namespace apic {

__device__ __forceinline__ int wrapN(int k, int n) { return (k + n) & (n - 1); }

__device__ __forceinline__ float zern_phase(const float* __restrict__ z, const float* c_sh, int nz) {
  float phi = 0.f;
  for (int j = 0; j < nz; ++j) phi += c_sh[j] * __ldg(&z[j]);
  return phi;
}

// ---------------------------------------------------------------- DF1: P_hat rows -> row IFFT
template <int N>
__global__ void __launch_bounds__(FftCfg<N>::THREADS)
df_build_p_rows(DevTables t, DarkDev L, const float2* __restrict__ O, const float* __restrict__ coef,
                float2* __restrict__ T, const int32_t* __restrict__ live_count, int chunk0) {
  extern __shared__ float2 sm[];
  __shared__ float c_sh[kMaxZern];
  const int slot = blockIdx.y, r0 = blockIdx.x * kLines;
  if (chunk0 + slot >= *live_count) return;
  if (threadIdx.x < t.nz) c_sh[threadIdx.x] = coef[size_t(slot) * t.nz + threadIdx.x];
  strip_zero<N>(sm);
  __syncthreads();
  const float2* o = O + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * L.d_ncol; idx += FftCfg<N>::THREADS) {
    const int l = idx / L.d_ncol, c = idx % L.d_ncol;
    if (r0 + l >= L.d_nrow) continue;
    const int fy = wrapN(L.d_row0 + r0 + l, N);
    const int e = L.dmap[fy * L.d_ncol + c];
    if (e < L.n_unknown) continue;                                     // not in P (unknown or outside)
    const int fx = wrapN(L.d_col0 + c, N);
    const float phi = zern_phase(L.zern + size_t(e) * t.nz, c_sh, t.nz);
    float sn, cs;
    sincosf(phi, &sn, &cs);
    strip_at<N>(sm, l, fx) = cmul(o[fy * N + fx], make_float2(cs, sn));
  }
  __syncthreads();
  fft_lines<N, true>(sm, t.tw);
  float2* tt = T + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
    const int l = idx / N, e = idx % N;
    if (r0 + l >= L.d_nrow) continue;
    tt[wrapN(L.d_row0 + r0 + l, N) * N + e] = strip_at<N>(sm, l, e);
  }
}

// ---------------------------------------------------------------- DF2: p, I - |p|^2, column FFT
template <int N>
__global__ void __launch_bounds__(FftCfg<N>::THREADS)
df_cols_p(DevTables t, DarkDev L, const float* __restrict__ d_int, float2* __restrict__ T, float2* __restrict__ PF,
          const int32_t* __restrict__ live, const int32_t* __restrict__ live_count, int chunk0) {
  extern __shared__ float2 sm[];
  const int slot = blockIdx.y, x0 = blockIdx.x * kLines;
  const int tile = resolve_tile_idx(live, live_count, chunk0, slot);
  if (tile < 0) return;
  strip_zero<N>(sm);
  __syncthreads();
  float2* tt = T + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * L.d_nrow; idx += FftCfg<N>::THREADS) {
    const int l = idx % kLines, r = idx / kLines;
    const int fy = wrapN(L.d_row0 + r, N);
    strip_at<N>(sm, l, fy) = tt[fy * N + x0 + l];
  }
  __syncthreads();
  fft_lines<N, true>(sm, t.tw);
  const float* img = d_int + (size_t(tile) * t.n_img + t.nb + L.led) * (N * N);
  float2* pf = PF + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
    const int l = idx % kLines, e = idx / kLines;
    float2& v = strip_at<N>(sm, l, e);
    const float2 p = v;
    pf[e * N + x0 + l] = p;
    v = make_float2(__ldg(&img[e * N + x0 + l]) - (p.x * p.x + p.y * p.y), 0.f);   // Eq. 13 lhs, spatial
  }
  __syncthreads();
  fft_lines<N, false>(sm, t.tw);
  for (int idx = threadIdx.x; idx < kLines * L.q_nrow; idx += FftCfg<N>::THREADS) {
    const int l = idx % kLines, r = idx / kLines;
    const int fy = wrapN(L.q_row0 + r, N);
    tt[fy * N + x0 + l] = strip_at<N>(sm, l, fy);
  }
}

// ---------------------------------------------------------------- DF3: row FFT, gather d on Q
template <int N>
__global__ void __launch_bounds__(FftCfg<N>::THREADS)
df_rows_rhs(DevTables t, DarkDev L, const float2* __restrict__ T, float2* __restrict__ vec_d, int max_eq,
            const int32_t* __restrict__ live_count, int chunk0) {
  extern __shared__ float2 sm[];
  const int slot = blockIdx.y, r0 = blockIdx.x * kLines;
  if (chunk0 + slot >= *live_count) return;
  const float2* tt = T + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
    const int l = idx / N, e = idx % N;
    float2 v = make_float2(0.f, 0.f);
    if (r0 + l < L.q_nrow) v = tt[wrapN(L.q_row0 + r0 + l, N) * N + e];
    strip_at<N>(sm, l, e) = v;
  }
  __syncthreads();
  fft_lines<N, false>(sm, t.tw);
  float2* d = vec_d + size_t(slot) * max_eq;
  const float scale = 1.f / float(N * N);
  for (int idx = threadIdx.x; idx < kLines * L.q_ncol; idx += FftCfg<N>::THREADS) {
    const int l = idx / L.q_ncol, c = idx % L.q_ncol;
    if (r0 + l >= L.q_nrow) continue;
    const int fy = wrapN(L.q_row0 + r0 + l, N);
    const int q = L.qmap[fy * L.q_ncol + c];
    if (q >= 0) d[q] = cscale(strip_at<N>(sm, l, wrapN(L.q_col0 + c, N)), scale);
  }
}

// ---------------------------------------------------------------- C: rows of Q
// FROM_VEC: scatter a Q-vector, row IFFT.  Otherwise: row FFT, keep Q only (x 1/N^2), row IFFT.
template <int N, bool FROM_VEC>
__global__ void __launch_bounds__(FftCfg<N>::THREADS)
df_rows_q(DevTables t, DarkDev L, float2* __restrict__ T, const float2* __restrict__ vec_d, int max_eq,
          const int32_t* __restrict__ cg_done, const int32_t* __restrict__ live_count, int chunk0) {
  extern __shared__ float2 sm[];
  const int slot = blockIdx.y, r0 = blockIdx.x * kLines;
  if (chunk0 + slot >= *live_count) return;
  if (!FROM_VEC && cg_done[slot]) return;
  float2* tt = T + size_t(slot) * (N * N);
  if (FROM_VEC) {
    strip_zero<N>(sm);
    __syncthreads();
    const float2* d = vec_d + size_t(slot) * max_eq;
    for (int idx = threadIdx.x; idx < kLines * L.q_ncol; idx += FftCfg<N>::THREADS) {
      const int l = idx / L.q_ncol, c = idx % L.q_ncol;
      if (r0 + l >= L.q_nrow) continue;
      const int fy = wrapN(L.q_row0 + r0 + l, N);
      const int q = L.qmap[fy * L.q_ncol + c];
      if (q >= 0) strip_at<N>(sm, l, wrapN(L.q_col0 + c, N)) = d[q];
    }
    __syncthreads();
  } else {
    for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
      const int l = idx / N, e = idx % N;
      float2 v = make_float2(0.f, 0.f);
      if (r0 + l < L.q_nrow) v = tt[wrapN(L.q_row0 + r0 + l, N) * N + e];
      strip_at<N>(sm, l, e) = v;
    }
    __syncthreads();
    fft_lines<N, false>(sm, t.tw);
    const float scale = 1.f / float(N * N);
    for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
      const int l = idx / N, fx = idx % N;
      float2& v = strip_at<N>(sm, l, fx);
      bool in = false;
      if (r0 + l < L.q_nrow) {
        const int kx = fx < N / 2 ? fx : fx - N;
        const int c = kx - L.q_col0;
        if (c >= 0 && c < L.q_ncol) in = L.qmap[wrapN(L.q_row0 + r0 + l, N) * L.q_ncol + c] >= 0;
      }
      v = in ? cscale(v, scale) : make_float2(0.f, 0.f);
    }
    __syncthreads();
  }
  fft_lines<N, true>(sm, t.tw);
  for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
    const int l = idx / N, e = idx % N;
    if (r0 + l >= L.q_nrow) continue;
    tt[wrapN(L.q_row0 + r0 + l, N) * N + e] = strip_at<N>(sm, l, e);
  }
}

// ---------------------------------------------------------------- B / D: column IFFT, . p or conj p, column FFT
template <int N, bool CONJ>
__global__ void __launch_bounds__(FftCfg<N>::THREADS)
df_cols_mul(DevTables t, float2* __restrict__ T, const float2* __restrict__ PF, int in_row0, int in_nrow,
            int out_row0, int out_nrow, const int32_t* __restrict__ cg_done, int check_done,
            const int32_t* __restrict__ live_count, int chunk0) {
  extern __shared__ float2 sm[];
  const int slot = blockIdx.y, x0 = blockIdx.x * kLines;
  if (chunk0 + slot >= *live_count) return;
  if (check_done && cg_done[slot]) return;
  strip_zero<N>(sm);
  __syncthreads();
  float2* tt = T + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * in_nrow; idx += FftCfg<N>::THREADS) {
    const int l = idx % kLines, r = idx / kLines;
    const int fy = wrapN(in_row0 + r, N);
    strip_at<N>(sm, l, fy) = tt[fy * N + x0 + l];
  }
  __syncthreads();
  fft_lines<N, true>(sm, t.tw);
  const float2* pf = PF + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
    const int l = idx % kLines, e = idx / kLines;
    float2& v = strip_at<N>(sm, l, e);
    const float2 p = pf[e * N + x0 + l];
    v = CONJ ? cmulc(v, p) : cmul(v, p);
  }
  __syncthreads();
  fft_lines<N, false>(sm, t.tw);
  for (int idx = threadIdx.x; idx < kLines * out_nrow; idx += FftCfg<N>::THREADS) {
    const int l = idx % kLines, r = idx / kLines;
    const int fy = wrapN(out_row0 + r, N);
    tt[fy * N + x0 + l] = strip_at<N>(sm, l, fy);
  }
}

// ---------------------------------------------------------------- A: E_U pdir, row IFFT
template <int N>
__global__ void __launch_bounds__(FftCfg<N>::THREADS)
df_rows_u_scatter(DevTables t, DarkDev L, float2* __restrict__ T, const float2* __restrict__ vec_p, int max_unknown,
                  const int32_t* __restrict__ cg_done, const int32_t* __restrict__ live_count, int chunk0) {
  extern __shared__ float2 sm[];
  const int slot = blockIdx.y, r0 = blockIdx.x * kLines;
  if (chunk0 + slot >= *live_count) return;
  if (cg_done[slot]) return;
  strip_zero<N>(sm);
  __syncthreads();
  const float2* pv = vec_p + size_t(slot) * max_unknown;
  for (int idx = threadIdx.x; idx < kLines * L.d_ncol; idx += FftCfg<N>::THREADS) {
    const int l = idx / L.d_ncol, c = idx % L.d_ncol;
    if (r0 + l >= L.u_nrow) continue;
    const int fy = wrapN(L.u_row0 + r0 + l, N);
    const int e = L.dmap[fy * L.d_ncol + c];
    if (e >= 0 && e < L.n_unknown) strip_at<N>(sm, l, wrapN(L.d_col0 + c, N)) = pv[e];
  }
  __syncthreads();
  fft_lines<N, true>(sm, t.tw);
  float2* tt = T + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
    const int l = idx / N, e = idx % N;
    if (r0 + l >= L.u_nrow) continue;
    tt[wrapN(L.u_row0 + r0 + l, N) * N + e] = strip_at<N>(sm, l, e);
  }
}

// ---------------------------------------------------------------- E: row FFT, gather U, partial <pdir, w>
template <int N>
__global__ void __launch_bounds__(FftCfg<N>::THREADS)
df_rows_u_gather(DevTables t, DarkDev L, const float2* __restrict__ T, float2* __restrict__ vec_w,
                 const float2* __restrict__ vec_p, int max_unknown, float* __restrict__ dot_part, int dot_parts,
                 const int32_t* __restrict__ cg_done, int check_done, const int32_t* __restrict__ live_count,
                 int chunk0) {
  extern __shared__ float2 sm[];
  __shared__ float red[FftCfg<N>::THREADS / 32];
  const int slot = blockIdx.y, r0 = blockIdx.x * kLines;
  if (chunk0 + slot >= *live_count) return;
  if (check_done && cg_done[slot]) return;
  const float2* tt = T + size_t(slot) * (N * N);
  for (int idx = threadIdx.x; idx < kLines * N; idx += FftCfg<N>::THREADS) {
    const int l = idx / N, e = idx % N;
    float2 v = make_float2(0.f, 0.f);
    if (r0 + l < L.u_nrow) v = tt[wrapN(L.u_row0 + r0 + l, N) * N + e];
    strip_at<N>(sm, l, e) = v;
  }
  __syncthreads();
  fft_lines<N, false>(sm, t.tw);
  float2* wv = vec_w + size_t(slot) * max_unknown;
  const float2* pv = vec_p + size_t(slot) * max_unknown;
  const float scale = 1.f / float(N * N);
  float dot = 0.f;
  for (int idx = threadIdx.x; idx < kLines * L.d_ncol; idx += FftCfg<N>::THREADS) {
    const int l = idx / L.d_ncol, c = idx % L.d_ncol;
    if (r0 + l >= L.u_nrow) continue;
    const int fy = wrapN(L.u_row0 + r0 + l, N);
    const int e = L.dmap[fy * L.d_ncol + c];
    if (e >= 0 && e < L.n_unknown) {
      const float2 w = cscale(strip_at<N>(sm, l, wrapN(L.d_col0 + c, N)), scale);
      wv[e] = w;
      if (check_done) {                       // inside the CG loop pdir is valid
        const float2 p = pv[e];
        dot += p.x * w.x + p.y * w.y;         // Re(conj(p) w)
      }
    }
  }
  for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = dot;
  __syncthreads();
  if (threadIdx.x == 0) {
    float s = 0.f;
    for (int i = 0; i < FftCfg<N>::THREADS / 32; ++i) s += red[i];
    dot_part[size_t(slot) * dot_parts + blockIdx.x] = s;
  }
}

// ---------------------------------------------------------------- F: CG vector updates (one CTA per tile)
__device__ __forceinline__ float block_sum_256(float v, float* red) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float s = 0.f;
  for (int i = 0; i < 8; ++i) s += red[i];
  return s;
}

// s = w (= C^H d), pdir = s, x = 0, gamma = gamma0 = ||s||^2
__global__ void __launch_bounds__(256) df_cg_init(int n_unknown, int max_unknown, float2* __restrict__ vec_x,
                                                  float2* __restrict__ vec_s, float2* __restrict__ vec_p,
                                                  const float2* __restrict__ vec_w, float* __restrict__ cg_scal,
                                                  int32_t* __restrict__ cg_done, int32_t* __restrict__ cg_iters,
                                                  int iters_ld, int led_pos, const int32_t* __restrict__ live_count,
                                                  int chunk0) {
  __shared__ float red[8];
  const int slot = blockIdx.x;
  if (chunk0 + slot >= *live_count) return;
  const size_t o = size_t(slot) * max_unknown;
  float g = 0.f;
  for (int e = threadIdx.x; e < n_unknown; e += 256) {
    const float2 s = vec_w[o + e];
    vec_s[o + e] = s;
    vec_p[o + e] = s;
    vec_x[o + e] = make_float2(0.f, 0.f);
    g += s.x * s.x + s.y * s.y;
  }
  g = block_sum_256(g, red);
  if (threadIdx.x == 0) {
    cg_scal[slot * 4 + 0] = g;
    cg_scal[slot * 4 + 1] = g;
    cg_done[slot] = !(g > 0.f);
    cg_iters[slot * iters_ld + led_pos] = 0;
  }
}

__global__ void __launch_bounds__(256) df_cg_update(int n_unknown, int max_unknown, float2* __restrict__ vec_x,
                                                    float2* __restrict__ vec_s, float2* __restrict__ vec_p,
                                                    const float2* __restrict__ vec_w, const float* __restrict__ dot_part,
                                                    int dot_parts, int n_parts, float* __restrict__ cg_scal,
                                                    int32_t* __restrict__ cg_done, int32_t* __restrict__ cg_iters,
                                                    int iters_ld, int led_pos, float tol2,
                                                    const int32_t* __restrict__ live_count, int chunk0) {
  __shared__ float red[8];
  const int slot = blockIdx.x;
  if (chunk0 + slot >= *live_count) return;
  if (cg_done[slot]) return;
  float pw = 0.f;
  for (int i = 0; i < n_parts; ++i) pw += dot_part[size_t(slot) * dot_parts + i];   // ||C pdir||^2
  const float gamma = cg_scal[slot * 4 + 0], gamma0 = cg_scal[slot * 4 + 1];
  if (!(pw > 0.f)) {
    if (threadIdx.x == 0) cg_done[slot] = 1;
    return;
  }
  const float alpha = gamma / pw;
  const size_t o = size_t(slot) * max_unknown;
  float g = 0.f;
  for (int e = threadIdx.x; e < n_unknown; e += 256) {
    const float2 p = vec_p[o + e], w = vec_w[o + e];
    float2 x = vec_x[o + e], s = vec_s[o + e];
    x.x += alpha * p.x; x.y += alpha * p.y;
    s.x -= alpha * w.x; s.y -= alpha * w.y;
    vec_x[o + e] = x;
    vec_s[o + e] = s;
    g += s.x * s.x + s.y * s.y;
  }
  g = block_sum_256(g, red);
  const float beta = g / gamma;
  for (int e = threadIdx.x; e < n_unknown; e += 256) {
    const float2 s = vec_s[o + e], p = vec_p[o + e];
    vec_p[o + e] = make_float2(s.x + beta * p.x, s.y + beta * p.y);
  }
  if (threadIdx.x == 0) {
    cg_scal[slot * 4 + 0] = g;
    cg_iters[slot * iters_ld + led_pos] += 1;
    if (!(g > tol2 * gamma0)) cg_done[slot] = 1;
  }
}

// ---------------------------------------------------------------- S10: O_hat(u) = U_hat(u) e^{-j phi(u+kappa)}
__global__ void __launch_bounds__(256) df_extend(DevTables t, DarkDev L, const float2* __restrict__ vec_x,
                                                 int max_unknown, const float* __restrict__ coef,
                                                 float2* __restrict__ O, const int32_t* __restrict__ live_count,
                                                 int chunk0) {
  __shared__ float c_sh[kMaxZern];
  const int slot = blockIdx.y;
  if (chunk0 + slot >= *live_count) return;
  if (threadIdx.x < t.nz) c_sh[threadIdx.x] = coef[size_t(slot) * t.nz + threadIdx.x];
  __syncthreads();
  const int e = blockIdx.x * 256 + threadIdx.x;
  if (e >= L.n_unknown) return;
  const float phi = zern_phase(L.zern + size_t(e) * t.nz, c_sh, t.nz);
  float sn, cs;
  sincosf(phi, &sn, &cs);
  O[size_t(slot) * t.n * t.n + L.disc_f[e]] = cmulc(vec_x[size_t(slot) * max_unknown + e], make_float2(cs, sn));
}

template <int N>
static void darkfield_led_n(const DevTables& t, const DarkDev& L, int led_pos, int n_dark_used, const Workspace& w,
                            const LaunchCtx& c, const float* d_int, int df_iters, float df_tol) {
  constexpr int TH = FftCfg<N>::THREADS;
  constexpr size_t SM = strip_smem_bytes(N);
  static bool attr = false;
  if (!attr) {
    const int sm = int(SM);
    cudaFuncSetAttribute(df_build_p_rows<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_cols_p<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_rows_rhs<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_rows_q<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_rows_q<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_cols_mul<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_cols_mul<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_rows_u_scatter<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_rows_u_gather<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    attr = true;
  }
  cudaStream_t s = c.stream;
  const int B = c.chunk_tiles;
  auto strips = [](int rows) { return (rows + kLines - 1) / kLines; };
  const dim3 g_d(strips(L.d_nrow), B), g_q(strips(L.q_nrow), B), g_u(strips(L.u_nrow), B), g_c(N / kLines, B);
  const int n_parts = strips(L.u_nrow);

#define APIC_LAUNCH(cat, ...) do { ProfScope ps_(c, cat); __VA_ARGS__; } while (0)
  APIC_LAUNCH(CAT_DF_BUILD_P_ROWS,
              (df_build_p_rows<N><<<g_d, TH, SM, s>>>(t, L, w.O, w.coef, w.T, c.live_count, c.chunk0)));
  APIC_LAUNCH(CAT_DF_COLS_P,
              (df_cols_p<N><<<g_c, TH, SM, s>>>(t, L, d_int, w.T, w.PF, c.live, c.live_count, c.chunk0)));
  APIC_LAUNCH(CAT_DF_ROWS_RHS,
              (df_rows_rhs<N><<<g_q, TH, SM, s>>>(t, L, w.T, w.vec_d, w.max_eq, c.live_count, c.chunk0)));
  // s0 = C^H d
  APIC_LAUNCH(CAT_DF_ROWS_Q, (df_rows_q<N, true><<<g_q, TH, SM, s>>>(t, L, w.T, w.vec_d, w.max_eq, w.cg_done,
                                                                     c.live_count, c.chunk0)));
  APIC_LAUNCH(CAT_DF_COLS_MUL,
              (df_cols_mul<N, false><<<g_c, TH, SM, s>>>(t, w.T, w.PF, L.q_row0, L.q_nrow, L.u_row0, L.u_nrow,
                                                         w.cg_done, 0, c.live_count, c.chunk0)));
  APIC_LAUNCH(CAT_DF_ROWS_U_GATHER,
              (df_rows_u_gather<N><<<g_u, TH, SM, s>>>(t, L, w.T, w.vec_w, w.vec_p, w.max_unknown, w.dot_part,
                                                       w.dot_parts, w.cg_done, 0, c.live_count, c.chunk0)));
  APIC_LAUNCH(CAT_DF_CG_VECTOR,
              (df_cg_init<<<B, 256, 0, s>>>(L.n_unknown, w.max_unknown, w.vec_x, w.vec_s, w.vec_p, w.vec_w, w.cg_scal,
                                            w.cg_done, w.cg_iters, n_dark_used, led_pos, c.live_count, c.chunk0)));
  const float tol2 = df_tol * df_tol;
  for (int it = 0; it < df_iters; ++it) {
    APIC_LAUNCH(CAT_DF_ROWS_U_SCATTER,
                (df_rows_u_scatter<N><<<g_u, TH, SM, s>>>(t, L, w.T, w.vec_p, w.max_unknown, w.cg_done, c.live_count,
                                                          c.chunk0)));
    APIC_LAUNCH(CAT_DF_COLS_MUL,
                (df_cols_mul<N, true><<<g_c, TH, SM, s>>>(t, w.T, w.PF, L.u_row0, L.u_nrow, L.q_row0, L.q_nrow,
                                                          w.cg_done, 1, c.live_count, c.chunk0)));
    APIC_LAUNCH(CAT_DF_ROWS_Q, (df_rows_q<N, false><<<g_q, TH, SM, s>>>(t, L, w.T, w.vec_d, w.max_eq, w.cg_done,
                                                                        c.live_count, c.chunk0)));
    APIC_LAUNCH(CAT_DF_COLS_MUL,
                (df_cols_mul<N, false><<<g_c, TH, SM, s>>>(t, w.T, w.PF, L.q_row0, L.q_nrow, L.u_row0, L.u_nrow,
                                                           w.cg_done, 1, c.live_count, c.chunk0)));
    APIC_LAUNCH(CAT_DF_ROWS_U_GATHER,
                (df_rows_u_gather<N><<<g_u, TH, SM, s>>>(t, L, w.T, w.vec_w, w.vec_p, w.max_unknown, w.dot_part,
                                                         w.dot_parts, w.cg_done, 1, c.live_count, c.chunk0)));
    APIC_LAUNCH(CAT_DF_CG_VECTOR,
                (df_cg_update<<<B, 256, 0, s>>>(L.n_unknown, w.max_unknown, w.vec_x, w.vec_s, w.vec_p, w.vec_w,
                                                w.dot_part, w.dot_parts, n_parts, w.cg_scal, w.cg_done, w.cg_iters,
                                                n_dark_used, led_pos, tol2, c.live_count, c.chunk0)));
  }
  APIC_LAUNCH(CAT_DF_EXTEND, (df_extend<<<dim3((L.n_unknown + 255) / 256, B), 256, 0, s>>>(
                                 t, L, w.vec_x, w.max_unknown, w.coef, w.O, c.live_count, c.chunk0)));
#undef APIC_LAUNCH
}

void launch_darkfield_led(const DevTables& t, const DarkDev& L, int led_pos, int n_dark_used, const Workspace& w,
                          const LaunchCtx& c, const float* d_int, int df_iters, float df_tol) {
  switch (t.n) {
    case 64: darkfield_led_n<64>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol); break;
    case 128: darkfield_led_n<128>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol); break;
    case 256: darkfield_led_n<256>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol); break;
    case 512: darkfield_led_n<512>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol); break;
  }
}

}  // namespace apic
