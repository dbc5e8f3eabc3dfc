// darkfield.cu - S8-S10 darkfield extension (Eq. 11-13; readings R15-R17, B1).
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
//
// Work is cut into strip TASKS (16 rows or 16 columns of one tile, fft_core.cuh); per tile the
// phases run in sequence:
//   setup   P0 build_p_rows -> P1 cols_p -> P2 rows_q -> P3 cols_mul(.p) -> P4 rows_u_gather -> P5 cg_init
//   iterate A rows_u_scatter -> B cols_mul(.conj p) -> C rows_q -> D cols_mul(.p) -> E rows_u_gather -> F cg_update
// Two schedulers run the same task bodies:
//   * persistent (default): ONE launch per LED and chunk; resident CTAs draw tasks from an atomic
//     ticket counter in phase-major order and wait on a per-tile progress counter, so tiles flow
//     through the phases independently (no grid-wide barrier, no host round trip; converged tiles
//     drop out, the launch ends when every tile has converged);
//   * multi-launch (df_mode 1): one kernel launch per phase, fixed df_iters iterations.
#include <algorithm>

#include "fft_core.cuh"
#include "plan.hpp"

namespace apic {

struct DfArgs {
  DevTables t;
  DarkDev L;
  const float* d_int;
  const float2* O_in;      // object spectrum (read in P0)
  float2* O;               // written by the final extension
  const float* coef;
  float2* T;
  float2* PF;
  float2 *vec_x, *vec_s, *vec_p, *vec_w;
  float* dot_part;
  float* cg_scal;
  int32_t* cg_done;
  int32_t* cg_iters;
  int max_unknown, dot_parts, iters_ld, led_pos;
  int max_iters;
  float tol2;
  const int32_t* live;
  const int32_t* live_count;
  int chunk0, n_tiles;
  // persistent scheduler state: [0] ticket, [1] tiles finished, [2 + slot] per-tile progress
  int32_t* sync;
  unsigned long long* work;   // executed nominal flop, 5 N log2 N per line transform (roofline line of bench.py)
};

__device__ __forceinline__ int wrapN(int k, int n) { return (k + n) & (n - 1); }
__device__ __forceinline__ float2 ldcg2(const float2* p) { return __ldcg(p); }

__device__ __forceinline__ float zern_phase(const float* __restrict__ z, const float* c_sh, int nz) {
  float phi = 0.f;
  for (int j = 0; j < nz; ++j) phi += c_sh[j] * __ldg(&z[j]);
  return phi;
}

template <int THREADS>
__device__ __forceinline__ float block_sum(float v, float* red) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float s = 0.f;
  for (int i = 0; i < THREADS / 32; ++i) s += red[i];
  return s;
}

// centred-row window test on an FFT-order row index
template <int N>
__device__ __forceinline__ bool in_rows(int fy, int row0, int nrow) {
  const int ky = fy < N / 2 ? fy : fy - N;
  return unsigned(ky - row0) < unsigned(nrow);
}
template <int N>
__device__ __forceinline__ int col_of(int fx, int col0) { return (fx < N / 2 ? fx : fx - N) - col0; }

// ---------------------------------------------------------------- P0: P_hat rows -> row IFFT
template <int N>
__device__ __forceinline__ void task_build_p_rows(const DfArgs& a, int slot, int strip, float2* sm, float* c_sh) {
  using S = Strip<N>;
  using TH = StripThread<N, false>;
  const DarkDev& L = a.L;
  const int nz = a.t.nz, line = TH::line(), tt = TH::t(), row = strip * S::LINES + line;
  __syncthreads();
  if (threadIdx.x < nz) c_sh[threadIdx.x] = a.coef[size_t(slot) * nz + threadIdx.x];
  __syncthreads();
  const bool valid = row < L.d_nrow;
  const int fy = wrapN(L.d_row0 + row, N);
  const float2* o = a.O_in + size_t(slot) * (N * N) + fy * N;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int fx = tt + S::TPL * r, c = col_of<N>(fx, L.d_col0);
    v[r] = make_float2(0.f, 0.f);
    if (valid && unsigned(c) < unsigned(L.d_ncol)) {
      const int e = __ldg(&L.dmap[fy * L.d_ncol + c]);
      if (e >= L.n_unknown) {                                          // in P = D_i ∩ known
        const float phi = zern_phase(L.zern + size_t(e) * nz, c_sh, nz);
        float sn, cs;
        sincosf(phi, &sn, &cs);
        v[r] = cmul(o[fx], make_float2(cs, sn));
      }
    }
  }
  fft_regs<N, true>(v, sm + line * S::LS, tt, a.t.tw);
  if (valid) {
    float2* tr = a.T + size_t(slot) * (N * N) + fy * N;
#pragma unroll
    for (int r = 0; r < S::R; ++r) tr[tt + S::TPL * r] = v[r];
  }
}

// ---------------------------------------------------------------- P1: p, I - |p|^2, column FFT
template <int N>
__device__ __forceinline__ void task_cols_p(const DfArgs& a, int slot, int tile, int strip, float2* sm) {
  using S = Strip<N>;
  using TH = StripThread<N, true>;
  const DarkDev& L = a.L;
  const int line = TH::line(), tt = TH::t(), x = strip * S::LINES + line;
  float2* tc = a.T + size_t(slot) * (N * N) + x;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int fy = tt + S::TPL * r;
    v[r] = in_rows<N>(fy, L.d_row0, L.d_nrow) ? ldcg2(&tc[fy * N]) : make_float2(0.f, 0.f);
  }
  fft_regs<N, true>(v, sm + line * S::LS, tt, a.t.tw);
  const float* img = a.d_int + (size_t(tile) * a.t.n_img + a.t.nb + L.led) * (N * N) + x;
  float2* pf = a.PF + size_t(slot) * (N * N) + x;
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int y = tt + S::TPL * r;
    const float2 p = v[r];
    pf[y * N] = p;
    v[r] = make_float2(__ldg(&img[y * N]) - (p.x * p.x + p.y * p.y), 0.f);       // Eq. 13 lhs, spatial
  }
  fft_regs<N, false>(v, sm + line * S::LS, tt, a.t.tw);
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int fy = tt + S::TPL * r;
    if (in_rows<N>(fy, L.q_row0, L.q_nrow)) tc[fy * N] = v[r];
  }
}

// ---------------------------------------------------------------- P2 / C: rows of Q
// row FFT, keep the bins of Q only (x 1/N^2), row IFFT.  In P2 this turns F(I-|p|^2) into M_Q d.
template <int N>
__device__ __forceinline__ void task_rows_q(const DfArgs& a, int slot, int strip, float2* sm) {
  using S = Strip<N>;
  using TH = StripThread<N, false>;
  const DarkDev& L = a.L;
  const int line = TH::line(), tt = TH::t(), row = strip * S::LINES + line;
  const bool valid = row < L.q_nrow;
  const int fy = wrapN(L.q_row0 + row, N);
  float2* tr = a.T + size_t(slot) * (N * N) + fy * N;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) v[r] = valid ? ldcg2(&tr[tt + S::TPL * r]) : make_float2(0.f, 0.f);
  fft_regs<N, false>(v, sm + line * S::LS, tt, a.t.tw);
  const float scale = 1.f / float(N * N);
  const int32_t* qrow = L.qmap + fy * L.q_ncol;
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int c = col_of<N>(tt + S::TPL * r, L.q_col0);
    const bool in = valid && unsigned(c) < unsigned(L.q_ncol) && __ldg(&qrow[c]) >= 0;
    v[r] = in ? cscale(v[r], scale) : make_float2(0.f, 0.f);
  }
  fft_regs<N, true>(v, sm + line * S::LS, tt, a.t.tw);
  if (valid) {
#pragma unroll
    for (int r = 0; r < S::R; ++r) tr[tt + S::TPL * r] = v[r];
  }
}

// ---------------------------------------------------------------- B / D / P3: column IFFT, . p or conj p, column FFT
template <int N, bool CONJ>
__device__ __forceinline__ void task_cols_mul(const DfArgs& a, int slot, int strip, float2* sm) {
  using S = Strip<N>;
  using TH = StripThread<N, true>;
  const DarkDev& L = a.L;
  const int in_row0 = CONJ ? L.u_row0 : L.q_row0, in_nrow = CONJ ? L.u_nrow : L.q_nrow;
  const int out_row0 = CONJ ? L.q_row0 : L.u_row0, out_nrow = CONJ ? L.q_nrow : L.u_nrow;
  const int line = TH::line(), tt = TH::t(), x = strip * S::LINES + line;
  float2* tc = a.T + size_t(slot) * (N * N) + x;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int fy = tt + S::TPL * r;
    v[r] = in_rows<N>(fy, in_row0, in_nrow) ? ldcg2(&tc[fy * N]) : make_float2(0.f, 0.f);
  }
  fft_regs<N, true>(v, sm + line * S::LS, tt, a.t.tw);
  const float2* pf = a.PF + size_t(slot) * (N * N) + x;
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const float2 p = ldcg2(&pf[(tt + S::TPL * r) * N]);
    v[r] = CONJ ? cmulc(v[r], p) : cmul(v[r], p);
  }
  fft_regs<N, false>(v, sm + line * S::LS, tt, a.t.tw);
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int fy = tt + S::TPL * r;
    if (in_rows<N>(fy, out_row0, out_nrow)) tc[fy * N] = v[r];
  }
}

// ---------------------------------------------------------------- A: E_U pdir, row IFFT
template <int N>
__device__ __forceinline__ void task_rows_u_scatter(const DfArgs& a, int slot, int strip, float2* sm) {
  using S = Strip<N>;
  using TH = StripThread<N, false>;
  const DarkDev& L = a.L;
  const int line = TH::line(), tt = TH::t(), row = strip * S::LINES + line;
  const bool valid = row < L.u_nrow;
  const int fy = wrapN(L.u_row0 + row, N);
  const float2* pv = a.vec_p + size_t(slot) * a.max_unknown;
  const int32_t* drow = L.dmap + fy * L.d_ncol;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int c = col_of<N>(tt + S::TPL * r, L.d_col0);
    v[r] = make_float2(0.f, 0.f);
    if (valid && unsigned(c) < unsigned(L.d_ncol)) {
      const int e = __ldg(&drow[c]);
      if (unsigned(e) < unsigned(L.n_unknown)) v[r] = ldcg2(&pv[e]);
    }
  }
  fft_regs<N, true>(v, sm + line * S::LS, tt, a.t.tw);
  if (valid) {
    float2* tr = a.T + size_t(slot) * (N * N) + fy * N;
#pragma unroll
    for (int r = 0; r < S::R; ++r) tr[tt + S::TPL * r] = v[r];
  }
}

// ---------------------------------------------------------------- E / P4: row FFT, gather U, partial <pdir, w>
template <int N>
__device__ __forceinline__ void task_rows_u_gather(const DfArgs& a, int slot, int strip, float2* sm, float* red,
                                                   bool with_dot) {
  using S = Strip<N>;
  using TH = StripThread<N, false>;
  const DarkDev& L = a.L;
  const int line = TH::line(), tt = TH::t(), row = strip * S::LINES + line;
  const bool valid = row < L.u_nrow;
  const int fy = wrapN(L.u_row0 + row, N);
  const float2* tr = a.T + size_t(slot) * (N * N) + fy * N;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) v[r] = valid ? ldcg2(&tr[tt + S::TPL * r]) : make_float2(0.f, 0.f);
  fft_regs<N, false>(v, sm + line * S::LS, tt, a.t.tw);
  float2* wv = a.vec_w + size_t(slot) * a.max_unknown;
  const float2* pv = a.vec_p + size_t(slot) * a.max_unknown;
  const int32_t* drow = L.dmap + fy * L.d_ncol;
  const float scale = 1.f / float(N * N);
  float dot = 0.f;
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int c = col_of<N>(tt + S::TPL * r, L.d_col0);
    if (valid && unsigned(c) < unsigned(L.d_ncol)) {
      const int e = __ldg(&drow[c]);
      if (unsigned(e) < unsigned(L.n_unknown)) {
        const float2 w = cscale(v[r], scale);
        wv[e] = w;
        if (with_dot) {
          const float2 p = ldcg2(&pv[e]);
          dot += p.x * w.x + p.y * w.y;         // Re(conj(p) w)
        }
      }
    }
  }
  dot = block_sum<S::THREADS>(dot, red);
  if (threadIdx.x == 0) a.dot_part[size_t(slot) * a.dot_parts + strip] = dot;
}

// ---------------------------------------------------------------- S10: O_hat(u) = U_hat(u) e^{-j phi(u+kappa)}
template <int THREADS>
__device__ __forceinline__ void extend_tile(const DfArgs& a, int slot, float* c_sh) {
  const DarkDev& L = a.L;
  const int nz = a.t.nz;
  __syncthreads();
  if (threadIdx.x < nz) c_sh[threadIdx.x] = a.coef[size_t(slot) * nz + threadIdx.x];
  __syncthreads();
  const float2* x = a.vec_x + size_t(slot) * a.max_unknown;
  float2* o = a.O + size_t(slot) * a.t.n * a.t.n;
  for (int e = threadIdx.x; e < L.n_unknown; e += THREADS) {
    const float phi = zern_phase(L.zern + size_t(e) * nz, c_sh, nz);
    float sn, cs;
    sincosf(phi, &sn, &cs);
    o[L.disc_f[e]] = cmulc(ldcg2(&x[e]), make_float2(cs, sn));
  }
}

// ---------------------------------------------------------------- P5: s = w (= C^H d), pdir = s, x = 0
// Returns true when the tile is already finished (zero right-hand side).
template <int THREADS>
__device__ __forceinline__ bool task_cg_init(const DfArgs& a, int slot, float* red) {
  const size_t o = size_t(slot) * a.max_unknown;
  float g = 0.f;
  for (int e = threadIdx.x; e < a.L.n_unknown; e += THREADS) {
    const float2 s = ldcg2(&a.vec_w[o + e]);
    a.vec_s[o + e] = s;
    a.vec_p[o + e] = s;
    a.vec_x[o + e] = make_float2(0.f, 0.f);
    g += s.x * s.x + s.y * s.y;
  }
  g = block_sum<THREADS>(g, red);
  const bool done = !(g > 0.f);
  if (threadIdx.x == 0) {
    a.cg_scal[slot * 4 + 0] = g;
    a.cg_scal[slot * 4 + 1] = g;
    a.cg_done[slot] = done;
    a.cg_iters[slot * a.iters_ld + a.led_pos] = 0;
  }
  return done;
}

// ---------------------------------------------------------------- F: CG vector updates
// Returns true when the tile has converged (||C^H r|| <= tol ||C^H d||) or cannot progress.
template <int THREADS>
__device__ __forceinline__ bool task_cg_update(const DfArgs& a, int slot, int n_parts, float* red) {
  float pw = 0.f;
  for (int i = 0; i < n_parts; ++i) pw += __ldcg(&a.dot_part[size_t(slot) * a.dot_parts + i]);   // ||C pdir||^2
  const float gamma = __ldcg(&a.cg_scal[slot * 4 + 0]), gamma0 = __ldcg(&a.cg_scal[slot * 4 + 1]);
  if (!(pw > 0.f)) {
    if (threadIdx.x == 0) a.cg_done[slot] = 1;
    return true;
  }
  const float alpha = gamma / pw;
  const size_t o = size_t(slot) * a.max_unknown;
  float g = 0.f;
  for (int e = threadIdx.x; e < a.L.n_unknown; e += THREADS) {
    const float2 p = ldcg2(&a.vec_p[o + e]), w = ldcg2(&a.vec_w[o + e]);
    float2 x = ldcg2(&a.vec_x[o + e]), s = ldcg2(&a.vec_s[o + e]);
    x.x += alpha * p.x; x.y += alpha * p.y;
    s.x -= alpha * w.x; s.y -= alpha * w.y;
    a.vec_x[o + e] = x;
    a.vec_s[o + e] = s;
    g += s.x * s.x + s.y * s.y;
  }
  g = block_sum<THREADS>(g, red);
  const float beta = g / gamma;
  for (int e = threadIdx.x; e < a.L.n_unknown; e += THREADS) {
    const float2 s = ldcg2(&a.vec_s[o + e]), p = ldcg2(&a.vec_p[o + e]);   // own writes: same thread, same e
    a.vec_p[o + e] = make_float2(s.x + beta * p.x, s.y + beta * p.y);
  }
  const bool done = !(g > a.tol2 * gamma0);
  if (threadIdx.x == 0) {
    a.cg_scal[slot * 4 + 0] = g;
    a.cg_iters[slot * a.iters_ld + a.led_pos] += 1;
    if (done) a.cg_done[slot] = 1;
  }
  return done;
}

// ================================================================ multi-launch scheduler (df_mode 1)
enum { PH_BUILD = 0, PH_COLS_P, PH_ROWS_Q, PH_COLS_MUL, PH_COLS_MUL_CONJ, PH_U_GATHER0, PH_U_GATHER, PH_U_SCATTER };

template <int N, int PHASE>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB) df_phase_kernel(DfArgs a, int check_done) {
  extern __shared__ float2 sm[];
  __shared__ float c_sh[kMaxZern];
  __shared__ float red[Strip<N>::THREADS / 32];
  const int slot = blockIdx.y, strip = blockIdx.x;
  const int tile = resolve_tile_idx(a.live, a.live_count, a.chunk0, slot);
  if (tile < 0) return;
  if (check_done && a.cg_done[slot]) return;
  if (PHASE == PH_BUILD) task_build_p_rows<N>(a, slot, strip, sm, c_sh);
  if (PHASE == PH_COLS_P) task_cols_p<N>(a, slot, tile, strip, sm);
  if (PHASE == PH_ROWS_Q) task_rows_q<N>(a, slot, strip, sm);
  if (PHASE == PH_COLS_MUL) task_cols_mul<N, false>(a, slot, strip, sm);
  if (PHASE == PH_COLS_MUL_CONJ) task_cols_mul<N, true>(a, slot, strip, sm);
  if (PHASE == PH_U_GATHER0) task_rows_u_gather<N>(a, slot, strip, sm, red, false);
  if (PHASE == PH_U_GATHER) task_rows_u_gather<N>(a, slot, strip, sm, red, true);
  if (PHASE == PH_U_SCATTER) task_rows_u_scatter<N>(a, slot, strip, sm);
}

// MODE 0: cg_init, 1: cg_update, 2: extend
template <int MODE>
__global__ void __launch_bounds__(256) df_vector_kernel(DfArgs a, int n_parts) {
  __shared__ float red[8];
  __shared__ float c_sh[kMaxZern];
  const int slot = blockIdx.x;
  if (a.chunk0 + slot >= *a.live_count) return;
  if (MODE == 0) task_cg_init<256>(a, slot, red);
  if (MODE == 1) { if (a.cg_done[slot]) return; task_cg_update<256>(a, slot, n_parts, red); }
  if (MODE == 2) extend_tile<256>(a, slot, c_sh);
}

// ================================================================ persistent scheduler (df_mode 0)
// Ticket order: setup phases P0..P5, then max_iters x (A..F); inside a phase tile-major.
struct Sched {
  int n[12];            // tasks per tile of P0..P5, A..F
  int cum[13];          // per-tile cumulative task count before each phase; cum[6] = setup total
  int lines[12];        // N-point line transforms executed by one task of each phase
};

template <int N>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB) df_persistent_kernel(DfArgs a, Sched sc) {
  constexpr int TH = Strip<N>::THREADS;
  extern __shared__ float2 sm[];
  __shared__ float c_sh[kMaxZern];
  __shared__ float red[TH / 32];
  __shared__ int sh_ticket, sh_stop, sh_skip;
  const int live_n = *a.live_count - a.chunk0;
  const int tiles = live_n < a.n_tiles ? live_n : a.n_tiles;
  if (tiles <= 0) return;
  const int setup_per_tile = sc.cum[6], iter_per_tile = sc.cum[12] - sc.cum[6];
  const long long setup_total = (long long)setup_per_tile * tiles;
  const long long iter_total = (long long)iter_per_tile * tiles;
  const long long total = setup_total + (long long)a.max_iters * iter_total;
  volatile int32_t* finished = a.sync + 1;
  volatile int32_t* prog = a.sync + 2;
  volatile int32_t* done_flag = a.cg_done;
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) {
      sh_ticket = atomicAdd(&a.sync[0], 1);
      sh_stop = (*finished >= tiles);
    }
    __syncthreads();
    const long long tk = sh_ticket;
    if (sh_stop || tk >= total) break;
    // ---- decode the ticket
    int ph, it = 0;
    long long r;
    if (tk < setup_total) {
      r = tk;
      ph = 0;
    } else {
      const long long q = tk - setup_total;
      it = int(q / iter_total);
      r = q % iter_total;
      ph = 6;
    }
    while (r >= (long long)sc.n[ph] * tiles) { r -= (long long)sc.n[ph] * tiles; ++ph; }
    const int slot = int(r / sc.n[ph]), strip = int(r % sc.n[ph]);
    const int need = sc.cum[ph] + it * iter_per_tile;                    // tasks of this tile to wait for
    // ---- wait for the tile's earlier phases (their tickets are lower, hence already drawn)
    if (threadIdx.x == 0) {
      while (prog[slot] < need && !(ph >= 6 && done_flag[slot])) __nanosleep(64);
      sh_skip = (ph >= 6 && done_flag[slot]);                            // tile converged earlier
      __threadfence();
    }
    __syncthreads();
    if (sh_skip) continue;
    bool tile_finished = false;
    switch (ph) {
      case 0: task_build_p_rows<N>(a, slot, strip, sm, c_sh); break;
      case 1: task_cols_p<N>(a, slot, a.live[a.chunk0 + slot], strip, sm); break;
      case 2: task_rows_q<N>(a, slot, strip, sm); break;
      case 3: task_cols_mul<N, false>(a, slot, strip, sm); break;
      case 4: task_rows_u_gather<N>(a, slot, strip, sm, red, false); break;
      case 5: tile_finished = task_cg_init<TH>(a, slot, red); break;
      case 6: task_rows_u_scatter<N>(a, slot, strip, sm); break;
      case 7: task_cols_mul<N, true>(a, slot, strip, sm); break;
      case 8: task_rows_q<N>(a, slot, strip, sm); break;
      case 9: task_cols_mul<N, false>(a, slot, strip, sm); break;
      case 10: task_rows_u_gather<N>(a, slot, strip, sm, red, true); break;
      default: {
        const bool conv = task_cg_update<TH>(a, slot, sc.n[10], red);
        tile_finished = conv || (it == a.max_iters - 1);
      } break;
    }
    if (tile_finished) extend_tile<TH>(a, slot, c_sh);                   // S10 for this tile
    // ---- publish: every thread fences its stores, then one thread bumps the tile's progress
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
      if (tile_finished) {
        done_flag[slot] = 1;
        __threadfence();
        atomicAdd(&a.sync[1], 1);
      }
      atomicAdd(&a.sync[2 + slot], 1);
      if (sc.lines[ph]) atomicAdd(a.work, (unsigned long long)sc.lines[ph] * (unsigned long long)(5 * N * (31 - __clz(N))));
    }
  }
}

template <int N>
static void darkfield_led_n(const DevTables& t, const DarkDev& L, int led_pos, int n_dark_used, const Workspace& w,
                            const LaunchCtx& c, const float* d_int, int df_iters, float df_tol, int df_mode) {
  constexpr int TH = Strip<N>::THREADS;
  constexpr int kLines = Strip<N>::LINES;
  constexpr size_t SM = Strip<N>::SMEM;
  static bool attr = false;
  static int resident = 0;
  if (!attr) {
    const int sm = int(SM);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_BUILD>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_COLS_P>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_ROWS_Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_COLS_MUL>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_COLS_MUL_CONJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_U_GATHER0>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_U_GATHER>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_phase_kernel<N, PH_U_SCATTER>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(df_persistent_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    int per_sm = 1, dev = 0, sms = 148;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, df_persistent_kernel<N>, TH, SM);
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    resident = (per_sm > 0 ? per_sm : 1) * sms;
    attr = true;
  }
  cudaStream_t s = c.stream;
  const int B = c.chunk_tiles;
  auto strips = [](int rows) { return (rows + kLines - 1) / kLines; };
  DfArgs a{};
  a.t = t; a.L = L; a.d_int = d_int; a.O_in = w.O; a.O = w.O; a.coef = w.coef; a.T = w.T; a.PF = w.PF;
  a.vec_x = w.vec_x; a.vec_s = w.vec_s; a.vec_p = w.vec_p; a.vec_w = w.vec_w;
  a.dot_part = w.dot_part; a.cg_scal = w.cg_scal; a.cg_done = w.cg_done; a.cg_iters = w.cg_iters;
  a.max_unknown = w.max_unknown; a.dot_parts = w.dot_parts; a.iters_ld = n_dark_used; a.led_pos = led_pos;
  a.max_iters = df_iters; a.tol2 = df_tol * df_tol;
  a.live = c.live; a.live_count = c.live_count; a.chunk0 = c.chunk0; a.n_tiles = B; a.sync = w.df_sync; a.work = w.df_work;
  const int n_d = strips(L.d_nrow), n_q = strips(L.q_nrow), n_u = strips(L.u_nrow), n_c = N / kLines;

  if (df_mode == 2) {
    Sched sc{};
    const int n[12] = {n_d, n_c, n_q, n_c, n_u, 1, n_u, n_c, n_q, n_c, n_u, 1};
    sc.cum[0] = 0;
    const int lines[12] = {1, 2, 2, 2, 1, 0, 1, 2, 2, 2, 1, 0};
    for (int i = 0; i < 12; ++i) { sc.n[i] = n[i]; sc.cum[i + 1] = sc.cum[i] + n[i]; sc.lines[i] = lines[i] * kLines; }
    cudaMemsetAsync(w.df_sync, 0, size_t(2 + w.chunk) * sizeof(int32_t), s);
    cudaMemsetAsync(w.cg_done, 0, size_t(w.chunk) * sizeof(int32_t), s);
    const long long widest = (long long)B * n_c;
    const int grid = int(std::min<long long>(resident, std::max<long long>(widest, 1)));
    ProfScope ps(c, CAT_DF_PERSISTENT);
    df_persistent_kernel<N><<<grid, TH, SM, s>>>(a, sc);
    return;
  }

#define APIC_LAUNCH(cat, ...) do { ProfScope ps_(c, cat); __VA_ARGS__; } while (0)
  const dim3 g_d(n_d, B), g_q(n_q, B), g_u(n_u, B), g_c(n_c, B);
  APIC_LAUNCH(CAT_DF_BUILD_P_ROWS, (df_phase_kernel<N, PH_BUILD><<<g_d, TH, SM, s>>>(a, 0)));
  APIC_LAUNCH(CAT_DF_COLS_P, (df_phase_kernel<N, PH_COLS_P><<<g_c, TH, SM, s>>>(a, 0)));
  APIC_LAUNCH(CAT_DF_ROWS_Q, (df_phase_kernel<N, PH_ROWS_Q><<<g_q, TH, SM, s>>>(a, 0)));
  APIC_LAUNCH(CAT_DF_COLS_MUL, (df_phase_kernel<N, PH_COLS_MUL><<<g_c, TH, SM, s>>>(a, 0)));
  APIC_LAUNCH(CAT_DF_ROWS_U_GATHER, (df_phase_kernel<N, PH_U_GATHER0><<<g_u, TH, SM, s>>>(a, 0)));
  APIC_LAUNCH(CAT_DF_CG_VECTOR, (df_vector_kernel<0><<<B, 256, 0, s>>>(a, n_u)));
  for (int it = 0; it < df_iters; ++it) {
    APIC_LAUNCH(CAT_DF_ROWS_U_SCATTER, (df_phase_kernel<N, PH_U_SCATTER><<<g_u, TH, SM, s>>>(a, 1)));
    APIC_LAUNCH(CAT_DF_COLS_MUL, (df_phase_kernel<N, PH_COLS_MUL_CONJ><<<g_c, TH, SM, s>>>(a, 1)));
    APIC_LAUNCH(CAT_DF_ROWS_Q, (df_phase_kernel<N, PH_ROWS_Q><<<g_q, TH, SM, s>>>(a, 1)));
    APIC_LAUNCH(CAT_DF_COLS_MUL, (df_phase_kernel<N, PH_COLS_MUL><<<g_c, TH, SM, s>>>(a, 1)));
    APIC_LAUNCH(CAT_DF_ROWS_U_GATHER, (df_phase_kernel<N, PH_U_GATHER><<<g_u, TH, SM, s>>>(a, 1)));
    APIC_LAUNCH(CAT_DF_CG_VECTOR, (df_vector_kernel<1><<<B, 256, 0, s>>>(a, n_u)));
  }
  APIC_LAUNCH(CAT_DF_EXTEND, (df_vector_kernel<2><<<B, 256, 0, s>>>(a, n_u)));
#undef APIC_LAUNCH
}

void launch_darkfield_led(const DevTables& t, const DarkDev& L, int led_pos, int n_dark_used, const Workspace& w,
                          const LaunchCtx& c, const float* d_int, int df_iters, float df_tol, int df_mode) {
  switch (t.n) {
    case 64: darkfield_led_n<64>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol, df_mode); break;
    case 128: darkfield_led_n<128>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol, df_mode); break;
    case 256: darkfield_led_n<256>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol, df_mode); break;
    case 512: darkfield_led_n<512>(t, L, led_pos, n_dark_used, w, c, d_int, df_iters, df_tol, df_mode); break;
  }
}

}  // namespace apic
