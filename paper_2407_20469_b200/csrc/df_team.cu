// df_team.cu - S8-S10 darkfield extension, "team" scheduler (df_mode 0, the default).
//
// Same mathematics as darkfield.cu (Eq. 11-13; readings R15-R17, B1): per
// darkfield LED, conjugate gradients on the normal equations of  C u = d  with C applied by pruned
// FFTs.  What differs is who does the work and how the phases are ordered:
//
//   * ONE launch per chunk covers all darkfield LEDs.  A *team* of G CTAs (a thread-block cluster,
//     G in {1,2,4,8}; one CTA per SM) owns a tile and walks it through every LED: setup phases
//     P0..P5, CG iterations A..F, extension.  Teams take tiles round-robin.
//   * Inside a phase the team's CTAs take strips (LINES rows or columns) round-robin; between
//     dependent phases the team meets at a hardware cluster barrier (release/acquire, ~0.2 us)
//     instead of global tickets, progress counters, fences and polling.  Data between a row pass
//     and a column pass still travels through the L2-resident scratch T.
//   * The CG vectors x, s, pdir live in shared memory of EVERY CTA of the team and are updated
//     redundantly (identical code on identical data -> bitwise identical), so the two dot products
//     of an iteration need no cross-CTA reduction and the convergence decision is uniform across
//     the team by construction; only w = C^H C pdir crosses CTAs (through L2).
//   * Loads of the next strip are issued before the second transform of the current one.
#include <algorithm>

#include "fft_core.cuh"
#include "plan.hpp"

namespace apic {

template <int N> struct TeamCfg;
// LINES lines per strip, MINB CTAs per SM (co-resident CTAs belong to different tiles, so one computes
// while the other waits on loads or on its team's barrier)
template <> struct TeamCfg<64>  { static constexpr int LINES = 32, MINB = 2; };   // 8 threads per line  -> 256 threads
template <> struct TeamCfg<128> { static constexpr int LINES = 8,  MINB = 2; };   // 32                  -> 256
template <> struct TeamCfg<256> { static constexpr int LINES = 16, MINB = 2; };   // 16                  -> 256
template <> struct TeamCfg<512> { static constexpr int LINES = 8,  MINB = 1; };   // 64                  -> 512

struct TeamArgs {
  DevTables t;
  const DarkDev* leds;     // device array, processing order
  int n_leds;
  ImgSrc src;
  float2* O;               // [chunk][N*N] object spectrum, extended in place
  const float* coef;       // [chunk][nz]
  float2* T;               // [chunk][N*N] transform scratch
  float2* PF;              // [chunk][N*N] p = F^-1 P_hat
  float2* vec_w;           // [chunk][max_unknown]
  int32_t* cg_iters;       // [chunk][n_leds]
  int max_unknown, max_iters;
  float tol2;
  const int32_t* live;
  const int32_t* live_count;
  int chunk0, n_tiles;
  unsigned long long* work;
};

namespace team {

__device__ __forceinline__ int wrapN(int k, int n) { return (k + n) & (n - 1); }
__device__ __forceinline__ unsigned cluster_rank() {
  unsigned r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ unsigned cluster_size() {
  unsigned r;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
  return r;
}
// All threads of all CTAs of the team.  Orders global-memory writes before it against reads after it.
__device__ __forceinline__ void team_sync(bool multi) {
  if (multi) {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
  } else {
    __syncthreads();
  }
}

template <int N>
__device__ __forceinline__ bool in_rows(int fy, int row0, int nrow) {
  const int ky = fy < N / 2 ? fy : fy - N;
  return unsigned(ky - row0) < unsigned(nrow);
}
template <int N>
__device__ __forceinline__ int col_of(int fx, int col0) { return (fx < N / 2 ? fx : fx - N) - col0; }

template <int THREADS>
__device__ __forceinline__ float block_sum(float v, float* red) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < THREADS / 32; ++i) s += red[i];
  return s;
}

// Shared-memory state of one CTA
template <int N>
struct Ctx {
  using S = Strip<N, TeamCfg<N>::LINES>;
  float2* sm;          // strip buffer [LINES][LS]
  const float2* tw;    // twiddles (shared)
  float2 *xs, *ss, *ps, *ws;   // CG vectors [max_unknown]
  float* c_sh;         // Zernike coefficients of the tile
  float* red;
  const DarkDev* L;    // current LED (shared copy)
};

}  // namespace team

namespace team {

template <int N> using TS = Strip<N, TeamCfg<N>::LINES>;
template <int N, bool COLS> using TT = StripThread<N, COLS, TeamCfg<N>::LINES>;

__device__ __forceinline__ float zern_phase(const float* __restrict__ z, const float* c_sh, int nz) {
  float phi = 0.f;
  for (int j = 0; j < nz; ++j) phi += c_sh[j] * __ldg(&z[j]);
  return phi;
}

// ---- strip loads / stores of the scratch T (cross-CTA data: always through L2)
template <int N>
__device__ __forceinline__ void load_col_strip(float2 (&v)[TS<N>::R], const float2* __restrict__ tc, int tt, int row0,
                                               int nrow) {
#pragma unroll
  for (int r = 0; r < TS<N>::R; ++r) {
    const int fy = tt + TS<N>::TPL * r;
    v[r] = in_rows<N>(fy, row0, nrow) ? __ldcg(&tc[fy * N]) : make_float2(0.f, 0.f);
  }
}
template <int N>
__device__ __forceinline__ void store_col_strip(const float2 (&v)[TS<N>::R], float2* __restrict__ tc, int tt, int row0,
                                                int nrow) {
#pragma unroll
  for (int r = 0; r < TS<N>::R; ++r) {
    const int fy = tt + TS<N>::TPL * r;
    if (in_rows<N>(fy, row0, nrow)) tc[fy * N] = v[r];
  }
}
template <int N>
__device__ __forceinline__ void load_row_strip(float2 (&v)[TS<N>::R], const float2* __restrict__ tr, int tt, bool valid) {
#pragma unroll
  for (int r = 0; r < TS<N>::R; ++r) v[r] = valid ? __ldcg(&tr[tt + TS<N>::TPL * r]) : make_float2(0.f, 0.f);
}

// ---------------------------------------------------------------- P0: P_hat rows -> row IFFT -> T
template <int N>
__device__ __noinline__ void phase_build_p_rows(const TeamArgs& a, const Ctx<N>& c, int slot, unsigned g, unsigned G) {
  using S = TS<N>;
  const DarkDev& L = *c.L;
  const int nz = a.t.nz, line = TT<N, false>::line(), tt = TT<N, false>::t();
  const int n_st = (L.d_nrow + S::LINES - 1) / S::LINES;
  for (int st = g; st < n_st; st += G) {
    const int row = st * S::LINES + line;
    const bool valid = row < L.d_nrow;
    const int fy = wrapN(L.d_row0 + row, N);
    const float2* o = a.O + size_t(slot) * (N * N) + fy * N;
    float2 v[S::R];
#pragma unroll
    for (int r = 0; r < S::R; ++r) {
      const int fx = tt + S::TPL * r, cc = col_of<N>(fx, L.d_col0);
      v[r] = make_float2(0.f, 0.f);
      if (valid && unsigned(cc) < unsigned(L.d_ncol)) {
        const int e = __ldg(&L.dmap[fy * L.d_ncol + cc]);
        if (e >= L.n_unknown) {                                          // in P = D_i ∩ known
          const float phi = zern_phase(L.zern + size_t(e) * nz, c.c_sh, nz);
          float sn, cs;
          sincosf(phi, &sn, &cs);
          v[r] = cmul(__ldcg(&o[fx]), make_float2(cs, sn));
        }
      }
    }
    fft_regs<N, true, true>(v, c.sm + line * S::LS, tt, c.tw);
    if (valid) {
      float2* tr = a.T + size_t(slot) * (N * N) + fy * N;
#pragma unroll
      for (int r = 0; r < S::R; ++r) tr[tt + S::TPL * r] = v[r];
    }
  }
}

// ---------------------------------------------------------------- P1: p, I - |p|^2, column FFT
template <int N>
__device__ __noinline__ void phase_cols_p(const TeamArgs& a, const Ctx<N>& c, int slot, int tile, unsigned g, unsigned G) {
  using S = TS<N>;
  const DarkDev& L = *c.L;
  const int line = TT<N, true>::line(), tt = TT<N, true>::t();
  constexpr int n_st = N / S::LINES;
  const size_t ii = size_t(tile) * a.t.n_img + a.t.nb + L.led;
  for (int st = g; st < n_st; st += G) {
    const int x = st * S::LINES + line;
    float2* tc = a.T + size_t(slot) * (N * N) + x;
    float2 v[S::R];
    float im[S::R];
    load_col_strip<N>(v, tc, tt, L.d_row0, L.d_nrow);
#pragma unroll
    for (int r = 0; r < S::R; ++r) im[r] = img_load(a.src, ii, N * N, (tt + S::TPL * r) * N + x);
    fft_regs<N, true, true>(v, c.sm + line * S::LS, tt, c.tw);
    float2* pf = a.PF + size_t(slot) * (N * N) + x;
#pragma unroll
    for (int r = 0; r < S::R; ++r) {
      const float2 p = v[r];
      pf[(tt + S::TPL * r) * N] = p;
      v[r] = make_float2(im[r] - (p.x * p.x + p.y * p.y), 0.f);          // Eq. 13 lhs, spatial
    }
    fft_regs<N, false, true>(v, c.sm + line * S::LS, tt, c.tw);
    store_col_strip<N>(v, tc, tt, L.q_row0, L.q_nrow);
  }
}

// ---------------------------------------------------------------- P2 / C: rows of Q: FFT, M_Q / N^2, IFFT
template <int N>
__device__ __noinline__ void phase_rows_q(const TeamArgs& a, const Ctx<N>& c, int slot, unsigned g, unsigned G) {
  using S = TS<N>;
  const DarkDev& L = *c.L;
  const int line = TT<N, false>::line(), tt = TT<N, false>::t();
  const int n_st = (L.q_nrow + S::LINES - 1) / S::LINES;
  const float scale = 1.f / float(N * N);
  float2* tbase = a.T + size_t(slot) * (N * N);
  for (int st = g; st < n_st; st += G) {
    const int row = st * S::LINES + line;
    const bool valid = row < L.q_nrow;
    const int fy = wrapN(L.q_row0 + row, N);
    float2 v[S::R];
    load_row_strip<N>(v, tbase + fy * N, tt, valid);
    const int32_t* qrow = L.qmap + fy * L.q_ncol;
    unsigned keep = 0;
#pragma unroll
    for (int r = 0; r < S::R; ++r) {
      const int cc = col_of<N>(tt + S::TPL * r, L.q_col0);
      if (valid && unsigned(cc) < unsigned(L.q_ncol) && __ldg(&qrow[cc]) >= 0) keep |= 1u << r;
    }
    fft_regs<N, false, true>(v, c.sm + line * S::LS, tt, c.tw);
#pragma unroll
    for (int r = 0; r < S::R; ++r) v[r] = (keep >> r & 1u) ? cscale(v[r], scale) : make_float2(0.f, 0.f);
    fft_regs<N, true, true>(v, c.sm + line * S::LS, tt, c.tw);
    if (valid) {
      float2* tr = tbase + fy * N;
#pragma unroll
      for (int r = 0; r < S::R; ++r) tr[tt + S::TPL * r] = v[r];
    }
  }
}

// ---------------------------------------------------------------- B / D / P3: column IFFT, . p or conj p, column FFT
template <int N, bool CONJ>
__device__ __noinline__ void phase_cols_mul(const TeamArgs& a, const Ctx<N>& c, int slot, unsigned g, unsigned G) {
  using S = TS<N>;
  const DarkDev& L = *c.L;
  const int in_row0 = CONJ ? L.u_row0 : L.q_row0, in_nrow = CONJ ? L.u_nrow : L.q_nrow;
  const int out_row0 = CONJ ? L.q_row0 : L.u_row0, out_nrow = CONJ ? L.q_nrow : L.u_nrow;
  const int line = TT<N, true>::line(), tt = TT<N, true>::t();
  constexpr int n_st = N / S::LINES;
  float2* tbase = a.T + size_t(slot) * (N * N);
  const float2* pbase = a.PF + size_t(slot) * (N * N);
  for (int st = g; st < n_st; st += G) {
    const int x = st * S::LINES + line;
    float2 v[S::R];
    load_col_strip<N>(v, tbase + x, tt, in_row0, in_nrow);
    {
      float2 p[S::R];
#pragma unroll
      for (int r = 0; r < S::R; ++r) p[r] = __ldcg(&pbase[(tt + S::TPL * r) * N + x]);
      fft_regs<N, true, true>(v, c.sm + line * S::LS, tt, c.tw);
#pragma unroll
      for (int r = 0; r < S::R; ++r) v[r] = CONJ ? cmulc(v[r], p[r]) : cmul(v[r], p[r]);
    }
    fft_regs<N, false, true>(v, c.sm + line * S::LS, tt, c.tw);
    store_col_strip<N>(v, tbase + x, tt, out_row0, out_nrow);
  }
}

// ---------------------------------------------------------------- A: E_U pdir (shared memory) -> row IFFT -> T
template <int N>
__device__ __noinline__ void phase_rows_u_scatter(const TeamArgs& a, const Ctx<N>& c, int slot, unsigned g, unsigned G) {
  using S = TS<N>;
  const DarkDev& L = *c.L;
  const int line = TT<N, false>::line(), tt = TT<N, false>::t();
  const int n_st = (L.u_nrow + S::LINES - 1) / S::LINES;
  for (int st = g; st < n_st; st += G) {
    const int row = st * S::LINES + line;
    const bool valid = row < L.u_nrow;
    const int fy = wrapN(L.u_row0 + row, N);
    const int32_t* drow = L.dmap + fy * L.d_ncol;
    float2 v[S::R];
#pragma unroll
    for (int r = 0; r < S::R; ++r) {
      const int cc = col_of<N>(tt + S::TPL * r, L.d_col0);
      v[r] = make_float2(0.f, 0.f);
      if (valid && unsigned(cc) < unsigned(L.d_ncol)) {
        const int e = __ldg(&drow[cc]);
        if (unsigned(e) < unsigned(L.n_unknown)) v[r] = c.ps[e];
      }
    }
    fft_regs<N, true, true>(v, c.sm + line * S::LS, tt, c.tw);
    if (valid) {
      float2* tr = a.T + size_t(slot) * (N * N) + fy * N;
#pragma unroll
      for (int r = 0; r < S::R; ++r) tr[tt + S::TPL * r] = v[r];
    }
  }
}

// ---------------------------------------------------------------- E / P4: T -> row FFT -> gather U -> w (global)
template <int N>
__device__ __noinline__ void phase_rows_u_gather(const TeamArgs& a, const Ctx<N>& c, int slot, unsigned g, unsigned G) {
  using S = TS<N>;
  const DarkDev& L = *c.L;
  const int line = TT<N, false>::line(), tt = TT<N, false>::t();
  const int n_st = (L.u_nrow + S::LINES - 1) / S::LINES;
  const float scale = 1.f / float(N * N);
  float2* wv = a.vec_w + size_t(slot) * a.max_unknown;
  for (int st = g; st < n_st; st += G) {
    const int row = st * S::LINES + line;
    const bool valid = row < L.u_nrow;
    const int fy = wrapN(L.u_row0 + row, N);
    float2 v[S::R];
    load_row_strip<N>(v, a.T + size_t(slot) * (N * N) + fy * N, tt, valid);
    const int32_t* drow = L.dmap + fy * L.d_ncol;
    int ent[S::R];
#pragma unroll
    for (int r = 0; r < S::R; ++r) {
      const int cc = col_of<N>(tt + S::TPL * r, L.d_col0);
      ent[r] = (valid && unsigned(cc) < unsigned(L.d_ncol)) ? __ldg(&drow[cc]) : -1;
    }
    fft_regs<N, false, true>(v, c.sm + line * S::LS, tt, c.tw);
#pragma unroll
    for (int r = 0; r < S::R; ++r)
      if (unsigned(ent[r]) < unsigned(L.n_unknown)) wv[ent[r]] = cscale(v[r], scale);
  }
}

// ---------------------------------------------------------------- P5: s = pdir = w (= C^H d), x = 0
// Every CTA of the team runs this on its own shared copies.  Returns gamma = ||s||^2.
template <int THREADS>
__device__ __forceinline__ float cg_init(const TeamArgs& a, float2* xs, float2* ss, float2* ps, float* red, int slot,
                                         int n_unknown) {
  const float2* wv = a.vec_w + size_t(slot) * a.max_unknown;
  float gsum = 0.f;
  for (int e = threadIdx.x; e < n_unknown; e += THREADS) {
    const float2 s = __ldcg(&wv[e]);
    ss[e] = s;
    ps[e] = s;
    xs[e] = make_float2(0.f, 0.f);
    gsum += s.x * s.x + s.y * s.y;
  }
  return block_sum<THREADS>(gsum, red);
}

// ---------------------------------------------------------------- F: CG update (redundant per CTA)
// Returns true when converged (||C^H r|| <= tol ||C^H d||) or when no progress is possible.
template <int THREADS>
__device__ __forceinline__ bool cg_update(const TeamArgs& a, float2* xs, float2* ss, float2* ps, float2* ws, float* red,
                                          int slot, int n_unknown, float& gamma, float gamma0) {
  const float2* wv = a.vec_w + size_t(slot) * a.max_unknown;
  float pw = 0.f;
  for (int e = threadIdx.x; e < n_unknown; e += THREADS) {
    const float2 w = __ldcg(&wv[e]), p = ps[e];
    ws[e] = w;
    pw += p.x * w.x + p.y * w.y;                                         // Re(conj(pdir) w) = ||C pdir||^2
  }
  pw = block_sum<THREADS>(pw, red);
  if (!(pw > 0.f)) return true;
  const float alpha = gamma / pw;
  float gsum = 0.f;
  for (int e = threadIdx.x; e < n_unknown; e += THREADS) {                // same thread <-> same e as above
    const float2 p = ps[e], w = ws[e];
    float2 x = xs[e], s = ss[e];
    x.x += alpha * p.x; x.y += alpha * p.y;
    s.x -= alpha * w.x; s.y -= alpha * w.y;
    xs[e] = x;
    ss[e] = s;
    gsum += s.x * s.x + s.y * s.y;
  }
  gsum = block_sum<THREADS>(gsum, red);
  const float beta = gsum / gamma;
  for (int e = threadIdx.x; e < n_unknown; e += THREADS) {
    const float2 s = ss[e], p = ps[e];
    ps[e] = make_float2(s.x + beta * p.x, s.y + beta * p.y);
  }
  gamma = gsum;
  return !(gsum > a.tol2 * gamma0);
}

}  // namespace team

// ================================================================ the kernel
template <int N>
__global__ void __launch_bounds__(Strip<N, TeamCfg<N>::LINES>::THREADS, TeamCfg<N>::MINB) df_team_kernel(TeamArgs a) {
  using namespace team;
  using S = TS<N>;
  constexpr int TH = S::THREADS;
  extern __shared__ float2 dyn[];
  __shared__ float c_sh[kMaxZern];
  __shared__ float red[TH / 32];
  __shared__ DarkDev Lsh;
  Ctx<N> c;
  c.sm = dyn;
  float2* tw_s = dyn + S::LINES * S::LS;
  c.tw = tw_s;
  c.xs = tw_s + S::TW_ENTRIES;
  c.ss = c.xs + a.max_unknown;
  c.ps = c.ss + a.max_unknown;
  c.ws = c.ps + a.max_unknown;
  c.c_sh = c_sh;
  c.red = red;
  c.L = &Lsh;
  const unsigned G = cluster_size(), g = cluster_rank();
  const bool multi = G > 1;
  const int team_id = blockIdx.x / G, n_teams = gridDim.x / G;
  for (int i = threadIdx.x; i < S::TW_ENTRIES; i += TH) tw_s[i] = a.t.tw[i];
  const int live_n = *a.live_count - a.chunk0;
  const int tiles = live_n < a.n_tiles ? live_n : a.n_tiles;
  const int nz = a.t.nz;
  unsigned long long lines = 0;     // line transforms executed by this CTA (thread 0's copy is reported)
  auto strips = [](int rows) { return (rows + S::LINES - 1) / S::LINES; };
  auto mine = [&](int n_st) { return (n_st > int(g)) ? (n_st - int(g) + int(G) - 1) / int(G) : 0; };

  for (int slot = team_id; slot < tiles; slot += n_teams) {
    const int tile = a.live[a.chunk0 + slot];
    __syncthreads();
    if (threadIdx.x < nz) c_sh[threadIdx.x] = a.coef[size_t(slot) * nz + threadIdx.x];
    for (int k = 0; k < a.n_leds; ++k) {
      __syncthreads();
      if (threadIdx.x < sizeof(DarkDev) / sizeof(int))
        reinterpret_cast<int*>(&Lsh)[threadIdx.x] = reinterpret_cast<const int*>(&a.leds[k])[threadIdx.x];
      __syncthreads();
      const int n_unknown = Lsh.n_unknown;
      const int n_d = strips(Lsh.d_nrow), n_q = strips(Lsh.q_nrow), n_u = strips(Lsh.u_nrow), n_c = N / S::LINES;
      // ---- setup: P_hat -> p -> d on Q -> s = C^H d
      phase_build_p_rows<N>(a, c, slot, g, G);
      team_sync(multi);
      phase_cols_p<N>(a, c, slot, tile, g, G);
      team_sync(multi);
      phase_rows_q<N>(a, c, slot, g, G);
      team_sync(multi);
      phase_cols_mul<N, false>(a, c, slot, g, G);
      team_sync(multi);
      phase_rows_u_gather<N>(a, c, slot, g, G);
      team_sync(multi);
      lines += (unsigned long long)(S::LINES) * (mine(n_d) + 2 * mine(n_c) + 2 * mine(n_q) + 2 * mine(n_c) + mine(n_u));
      float gamma = cg_init<TH>(a, c.xs, c.ss, c.ps, red, slot, n_unknown);
      const float gamma0 = gamma;
      int iters = 0;
      bool done = !(gamma > 0.f);
      // ---- CG on the normal equations
      while (!done && iters < a.max_iters) {
        __syncthreads();                                   // pdir complete in shared memory
        phase_rows_u_scatter<N>(a, c, slot, g, G);
        team_sync(multi);
        phase_cols_mul<N, true>(a, c, slot, g, G);
        team_sync(multi);
        phase_rows_q<N>(a, c, slot, g, G);
        team_sync(multi);
        phase_cols_mul<N, false>(a, c, slot, g, G);
        team_sync(multi);
        phase_rows_u_gather<N>(a, c, slot, g, G);
        team_sync(multi);
        lines += (unsigned long long)(S::LINES) * (mine(n_u) + 2 * mine(n_c) + 2 * mine(n_q) + 2 * mine(n_c) + mine(n_u));
        done = cg_update<TH>(a, c.xs, c.ss, c.ps, c.ws, red, slot, n_unknown, gamma, gamma0);
        ++iters;
      }
      __syncthreads();
      // ---- S10: O_hat(u) = U_hat(u) e^{-j phi(u+kappa)}, known ∪= U (entries split over the team)
      {
        float2* o = a.O + size_t(slot) * (N * N);
        for (int e = int(g) * TH + threadIdx.x; e < n_unknown; e += int(G) * TH) {
          const float phi = zern_phase(Lsh.zern + size_t(e) * nz, c_sh, nz);
          float sn, cs;
          sincosf(phi, &sn, &cs);
          const int q = Lsh.disc_f[e];
          const float2 u = cmulc(c.xs[e], make_float2(cs, sn));
          o[q] = Lsh.accumulate ? cadd(__ldcg(&o[q]), u) : u;   // ring-wise order (R15b): sum now, mean at the end of the ring
        }
        if (g == 0 && threadIdx.x == 0) a.cg_iters[size_t(slot) * a.n_leds + k] = iters;
      }
      team_sync(multi);                                    // O complete before the next LED reads it
      if (Lsh.n_avg > 0) {                                 // df_order 1, end of a ring: bins solved by c LEDs hold a sum of c solutions
        float2* o = a.O + size_t(slot) * (N * N);
        for (int i = int(g) * TH + threadIdx.x; i < Lsh.n_avg; i += int(G) * TH) {
          const int q = __ldg(&Lsh.avg_f[i]);
          o[q] = cscale(__ldcg(&o[q]), __ldg(&Lsh.avg_w[i]));
        }
        team_sync(multi);
      }
    }
  }
  // reported as nominal flop: 5 N log2 N per N-point line transform
  if (threadIdx.x == 0 && lines) atomicAdd(a.work, lines * (unsigned long long)(5 * N * (31 - __clz(N))));
}

template <int N>
static void darkfield_team_n(const DevTables& t, const DarkDev* d_leds, int n_leds, const Workspace& w,
                             const LaunchCtx& c, const ImgSrc& src, int df_iters, float df_tol, int team_size) {
  using S = Strip<N, TeamCfg<N>::LINES>;
  const size_t smem = (size_t(S::LINES) * S::LS + S::TW_ENTRIES + 4 * size_t(w.max_unknown)) * sizeof(float2);
  const int sms = c.pd->sms;
  int per_sm = 1;
  if (!c.pd->attr_team) {
    cudaFuncSetAttribute(df_team_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 4096);
    cudaFuncSetAttribute(df_team_kernel<N>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    c.pd->attr_team = true;
  }
  TeamArgs a{};
  a.t = t; a.leds = d_leds; a.n_leds = n_leds; a.src = src; a.O = w.O; a.coef = w.coef; a.T = w.T; a.PF = w.PF;
  a.vec_w = w.vec_w; a.cg_iters = w.cg_iters; a.max_unknown = w.max_unknown; a.max_iters = df_iters;
  a.tol2 = df_tol * df_tol; a.live = c.live; a.live_count = c.live_count; a.chunk0 = c.chunk0;
  a.n_tiles = c.chunk_tiles; a.work = w.df_work;
  // team size: as many CTAs per tile as the chunk leaves SMs for (power of two, <= 8)
  int G = team_size;
  if (G <= 0) {
    G = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, df_team_kernel<N>, S::THREADS, smem);
    per_sm = std::max(1, per_sm);
    while (G < 8 && 2 * G * c.chunk_tiles <= sms * per_sm) G *= 2;
    if (N >= 512 && G < 4) G = 4;                      // keep the per-team working set of the chunk inside L2
  }
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = unsigned(G); at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3(S::THREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = c.stream;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  int max_clusters = 0;
  cfg.gridDim = dim3(unsigned(G) * unsigned(sms / G));
  if (cudaOccupancyMaxActiveClusters(&max_clusters, df_team_kernel<N>, &cfg) != cudaSuccess || max_clusters < 1)
    max_clusters = std::max(1, sms / G - (G > 2 ? 2 : 0));
  const int teams = std::max(1, std::min(max_clusters, c.chunk_tiles));
  cfg.gridDim = dim3(unsigned(G) * unsigned(teams));
  ProfScope ps(c, CAT_DF_TEAM);
  cudaLaunchKernelEx(&cfg, df_team_kernel<N>, a);
}

void launch_darkfield_team(const DevTables& t, const DarkDev* d_leds, int n_leds, const Workspace& w, const LaunchCtx& c,
                           const ImgSrc& src, int df_iters, float df_tol, int team_size) {
  if (n_leds <= 0) return;
  switch (t.n) {
    case 64: darkfield_team_n<64>(t, d_leds, n_leds, w, c, src, df_iters, df_tol, team_size); break;
    case 128: darkfield_team_n<128>(t, d_leds, n_leds, w, c, src, df_iters, df_tol, team_size); break;
    case 256: darkfield_team_n<256>(t, d_leds, n_leds, w, c, src, df_iters, df_tol, team_size); break;
    case 512: darkfield_team_n<512>(t, d_leds, n_leds, w, c, src, df_iters, df_tol, team_size); break;
  }
}

}  // namespace apic
