// df_mgrid.cu - S8-S10 darkfield extension on per-LED reduced cyclic grids (df_mode 0 at N = 256).
//
// Same mathematics as df_team.cu (Eq. 11-13; readings R15-R17, B1): per darkfield
// LED, conjugate gradients on the normal equations of  C u = d,  C[k,u] = conj P_hat(u - k), k in Q,
// u in U, with C and C^H applied by FFTs.  What is new is the grid those FFTs run on.  C u only
// needs the cross-correlation of u (supported on U) with P_hat (supported on P) at the lags k in Q,
// and C^H r the correlation of r (on Q) with P_hat at the lags in U.  On a cyclic grid of mx x my
// bins the wrong pairs are those with  u - p - k = (a mx, b my) != 0,  so the grid is alias-free as
// soon as mx, my exceed the extent of U - P - Q along each axis (geometry.cpp picks mx, my from
// {96,128,160,192,256} per LED; e.g. 96 x 160 or 128 x 160 for config 2 instead of 256 x 256).
// p is then sampled on that grid (p_M = F_M^-1 P_hat): 3-4x fewer points per transform.  Only the
// right-hand side d = F(I - |p|^2)/N^2 (Eq. 13) needs the N x N grid, once per LED.
//
// Scheduling is df_team.cu's: one launch per pass covers every LED; a thread-block cluster (team)
// owns a tile, its CTAs split the 16-line strips of each phase and meet at cluster barriers; the CG
// vectors live redundantly in every CTA's shared memory.  Line transforms are fft_xy.cuh's X/Y pair.
#include <algorithm>
#include <type_traits>

#include "fft_xy.cuh"
#include "plan.hpp"

namespace apic {
namespace mg {

constexpr int N = 256;
constexpr int TH = 256;
using S256 = Strip<256>;     // N-grid line transform of fft_core.cuh (16 lines x 16 threads)

struct Args {
  DevTables t;
  const DarkDev* leds;
  int n_leds;
  ImgSrc src;
  float2* O;               // [chunk][N*N] object spectrum, extended in place
  const float* coef;       // [chunk][nz]
  float2* T;               // [chunk][N*N] N-grid scratch (right-hand side only)
  float2* TM;              // [chunk][N*N] reduced-grid scratch
  float2* PF;              // [chunk][N*N] p_M = F_M^-1 P_hat
  float2* vec_w;           // [chunk][max_unknown]
  int32_t* cg_iters;
  int max_unknown, max_iters;
  float tol2;
  const int32_t* live;
  const int32_t* live_count;
  int chunk0, n_tiles;
  unsigned long long* work;   // executed nominal flop (5 L log2 L per line transform)
};

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
__device__ __forceinline__ void team_sync(bool multi) {
  if (multi) {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
  } else {
    __syncthreads();
  }
}
__device__ __forceinline__ float block_sum(float v, float* red) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < TH / 32; ++i) s += red[i];
  return s;
}
__device__ __forceinline__ int modp(int k, int m) {   // k mod m for k in (-m, m)... generalised
  int r = k % m;
  return r < 0 ? r + m : r;
}
// is grid row g (0 <= g < m) one of the nrow rows starting at centred row row0 (mod m)?
__device__ __forceinline__ bool row_in(int g, int row0m, int nrow, int m) {
  int d = g - row0m;
  if (d < 0) d += m;
  return d < nrow;
}
__device__ __forceinline__ float zern_phase(const float* __restrict__ z, const float* c_sh, int nz) {
  float phi = 0.f;
  for (int j = 0; j < nz; ++j) phi += c_sh[j] * __ldg(&z[j]);
  return phi;
}
__host__ __device__ constexpr int tw_slot(int r1) { return r1 == 6 ? 0 : r1 == 8 ? 1 : r1 == 10 ? 2 : r1 == 12 ? 3 : 4; }
__host__ __device__ inline double line_flop(int L) { return 5.0 * L * log2(double(L)); }

// calls f(std::integral_constant<int, R1>) for the run-time r1
template <class F>
__device__ __forceinline__ void with_r1(int r1, F&& f) {
  switch (r1) {
    case 6: f(std::integral_constant<int, 6>()); break;
    case 8: f(std::integral_constant<int, 8>()); break;
    case 10: f(std::integral_constant<int, 10>()); break;
    case 12: f(std::integral_constant<int, 12>()); break;
    default: f(std::integral_constant<int, 16>()); break;
  }
}

// Shared-memory layout of a CTA (all dynamic, so that every access is an LDS/STS and no generic LD/ST):
//   [bufA kXyBuf][bufB kXyBuf][twx 256][twy 256][tw256 256][misc 128][xs mu][ss mu][ps mu]   (float2 units)
// misc: Zernike coefficients of the tile (64 floats), block_sum scratch (8 floats), the current DarkDev.
struct Ctx {
  int mu;   // max_unknown
  __device__ __forceinline__ float2* base() const {
    extern __shared__ float2 dyn[];
    return dyn;
  }
  __device__ __forceinline__ float2* bufA() const { return base(); }
  __device__ __forceinline__ float2* bufB() const { return base() + kXyBuf; }
  __device__ __forceinline__ float2* twx() const { return base() + 2 * kXyBuf; }
  __device__ __forceinline__ float2* twy() const { return base() + 2 * kXyBuf + 256; }
  __device__ __forceinline__ float2* tw256() const { return base() + 2 * kXyBuf + 512; }
  __device__ __forceinline__ float* c_sh() const { return reinterpret_cast<float*>(base() + 2 * kXyBuf + 768); }
  __device__ __forceinline__ float* red() const { return c_sh() + 64; }
  __device__ __forceinline__ DarkDev* Lp() const { return reinterpret_cast<DarkDev*>(c_sh() + 80); }
  __device__ __forceinline__ float2* xs() const { return base() + 2 * kXyBuf + 768 + 128; }
  __device__ __forceinline__ float2* ss() const { return xs() + mu; }
  __device__ __forceinline__ float2* ps() const { return ss() + mu; }
};
constexpr int kSmFixed = 2 * kXyBuf + 768 + 128;   // float2 entries before the CG vectors
static_assert(sizeof(DarkDev) <= (256 - 80) * sizeof(float), "DarkDev does not fit the misc region");
static_assert(kMaxZern <= 64, "c_sh region");

// ================================================================ reduced-grid phases
// A: E_U pdir (shared memory) -> row IFFT_mx -> TM rows of U
template <int R1>
__device__ __noinline__ void ph_rows_u_scatter(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.u_nrow + 15) >> 4;
  float2* tm = a.TM + size_t(slot) * (N * N);
  int par = 0;
  for (int st = g; st < n_st; st += G, par ^= 1) {
    float2 v[16];
    {
      const int row = st * 16 + M::a_line(), t = M::a_t();
      const int32_t* drow = L.dmap_m + modp(L.u_row0 + row, my) * mx;
#pragma unroll
      for (int r = 0; r < R1; ++r) {
        v[r] = make_float2(0.f, 0.f);
        if (row < L.u_nrow) {
          const int e = __ldg(&drow[t + 16 * r]);
          if (unsigned(e) < unsigned(L.n_unknown)) v[r] = c.ps()[e];
        }
      }
    }
    fft_x<R1, true, false>(v, par ? c.bufB() : c.bufA(), c.twx());
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.u_nrow) {
        float2* tr = tm + modp(L.u_row0 + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) tr[R1 * k2] = v[k2];
      }
    }
  }
}

// E: TM rows of U -> row FFT_mx -> gather U -> w / (mx my)
template <int R1>
__device__ __noinline__ void ph_rows_u_gather(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.u_nrow + 15) >> 4;
  const float scale = 1.f / float(mx * my);
  const float2* tm = a.TM + size_t(slot) * (N * N);
  float2* wv = a.vec_w + size_t(slot) * a.max_unknown;
  int par = 0;
  for (int st = g; st < n_st; st += G, par ^= 1) {
    float2 v[16];
    {
      const int row = st * 16 + M::a_line(), t = M::a_t();
      const float2* tr = tm + modp(L.u_row0 + row, my) * mx + t;
#pragma unroll
      for (int r = 0; r < R1; ++r) v[r] = row < L.u_nrow ? __ldcg(&tr[16 * r]) : make_float2(0.f, 0.f);
    }
    fft_x<R1, false, false>(v, par ? c.bufB() : c.bufA(), c.twx());
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.u_nrow) {
        const int32_t* drow = L.dmap_m + modp(L.u_row0 + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const int e = __ldg(&drow[R1 * k2]);
          if (unsigned(e) < unsigned(L.n_unknown)) wv[e] = cscale(v[k2], scale);
        }
      }
    }
  }
}

// C: TM rows of Q: row FFT_mx, M_Q / (mx my), row IFFT_mx
template <int R1>
__device__ __noinline__ void ph_rows_q(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.q_nrow + 15) >> 4;
  const float scale = 1.f / float(mx * my);
  float2* tm = a.TM + size_t(slot) * (N * N);
  for (int st = g; st < n_st; st += G) {
    float2 v[16];
    const int rowa = st * 16 + M::a_line(), t = M::a_t();
    float2* tr = tm + modp(L.q_row0 + rowa, my) * mx + t;
#pragma unroll
    for (int r = 0; r < R1; ++r) v[r] = rowa < L.q_nrow ? __ldcg(&tr[16 * r]) : make_float2(0.f, 0.f);
    unsigned keep = 0;
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.q_nrow) {
        const uint8_t* qrow = L.qmask_m + modp(L.q_row0 + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) keep |= unsigned(__ldg(&qrow[R1 * k2]) != 0) << k2;
      }
    }
    fft_x<R1, false, false>(v, c.bufA(), c.twx());
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) v[k2] = (keep >> k2 & 1u) ? cscale(v[k2], scale) : make_float2(0.f, 0.f);
    fft_y<R1, true, false>(v, c.bufB(), c.twx());
    if (rowa < L.q_nrow) {
#pragma unroll
      for (int r = 0; r < R1; ++r) tr[16 * r] = v[r];
    }
  }
}

// B / D: TM columns: IFFT_my, . conj p_M (B) or . p_M (D), FFT_my
template <int R1, bool CONJ>
__device__ __noinline__ void ph_cols_mul(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  using M = XY<R1, true>;
  const DarkDev& L = *c.Lp();
  constexpr int my = 16 * R1;
  const int mx = L.mx, n_st = mx >> 4;
  const int in0 = modp(CONJ ? L.u_row0 : L.q_row0, my), in_n = CONJ ? L.u_nrow : L.q_nrow;
  const int out0 = modp(CONJ ? L.q_row0 : L.u_row0, my), out_n = CONJ ? L.q_nrow : L.u_nrow;
  float2* tm = a.TM + size_t(slot) * (N * N);
  const float2* pf = a.PF + size_t(slot) * (N * N);
  for (int st = g; st < n_st; st += G) {
    const int x = st * 16 + M::a_line(), t = M::a_t();
    float2 v[16], p[16];
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      v[r] = row_in(gy, in0, in_n, my) ? __ldcg(&tm[gy * mx + x]) : make_float2(0.f, 0.f);
    }
    if (M::b_active()) {
      const float2* pc = pf + M::b_k1() * mx + x;
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) p[k2] = __ldcg(&pc[(R1 * k2) * mx]);
    }
    fft_x<R1, true, true>(v, c.bufA(), c.twy());
    if (M::b_active()) {
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) v[k2] = CONJ ? cmulc(v[k2], p[k2]) : cmul(v[k2], p[k2]);
    }
    fft_y<R1, false, true>(v, c.bufB(), c.twy());
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      if (row_in(gy, out0, out_n, my)) tm[gy * mx + x] = v[r];
    }
  }
}

// ================================================================ setup phases
__device__ __forceinline__ int wrapN(int k) { return (k + N) & (N - 1); }
__device__ __forceinline__ float2 p_hat_entry(const Args& a, const Ctx& c, const float2* __restrict__ o, int e) {
  // P_hat(k) = O_hat(k) e^{+j phi(k + kappa)} on P = D_i ∩ known
  const DarkDev& L = *c.Lp();
  const float phi = zern_phase(L.zern + size_t(e) * a.t.nz, c.c_sh(), a.t.nz);
  float sn, cs;
  sincosf(phi, &sn, &cs);
  return cmul(__ldcg(&o[__ldg(&L.disc_f[e])]), make_float2(cs, sn));
}

// P0 (N grid): P_hat rows -> row IFFT_N -> T
__device__ __noinline__ void ph_build_p_rows_n(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  const DarkDev& L = *c.Lp();
  const int line = int(threadIdx.x) >> 4, tt = int(threadIdx.x) & 15;
  const int n_st = (L.d_nrow + 15) >> 4;
  const float2* o = a.O + size_t(slot) * (N * N);
  for (int st = g; st < n_st; st += G) {
    const int row = st * 16 + line;
    const bool valid = row < L.d_nrow;
    const int fy = wrapN(L.d_row0 + row);
    float2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int fx = tt + 16 * r, cc = (fx < N / 2 ? fx : fx - N) - L.d_col0;
      v[r] = make_float2(0.f, 0.f);
      if (valid && unsigned(cc) < unsigned(L.d_ncol)) {
        const int e = __ldg(&L.dmap[fy * L.d_ncol + cc]);
        if (e >= L.n_unknown) v[r] = p_hat_entry(a, c, o, e);
      }
    }
    fft_regs<N, true, true>(v, c.bufA() + line * S256::LS, tt, c.tw256());
    if (valid) {
      float2* tr = a.T + size_t(slot) * (N * N) + fy * N;
#pragma unroll
      for (int r = 0; r < 16; ++r) tr[tt + 16 * r] = v[r];
    }
  }
}

// P0' (reduced grid): P_hat rows -> row IFFT_mx -> TM
template <int R1>
__device__ __noinline__ void ph_build_p_rows_m(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.d_nrow + 15) >> 4;
  const float2* o = a.O + size_t(slot) * (N * N);
  float2* tm = a.TM + size_t(slot) * (N * N);
  int par = 0;
  __syncthreads();                                     // bufA was used by the N-grid transform
  for (int st = g; st < n_st; st += G, par ^= 1) {
    float2 v[16];
    {
      const int row = st * 16 + M::a_line(), t = M::a_t();
      const int32_t* drow = L.dmap_m + modp(L.d_row0 + row, my) * mx;
#pragma unroll
      for (int r = 0; r < R1; ++r) {
        v[r] = make_float2(0.f, 0.f);
        if (row < L.d_nrow) {
          const int e = __ldg(&drow[t + 16 * r]);
          if (e >= L.n_unknown) v[r] = p_hat_entry(a, c, o, e);
        }
      }
    }
    fft_x<R1, true, false>(v, par ? c.bufB() : c.bufA(), c.twx());
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.d_nrow) {
        float2* tr = tm + modp(L.d_row0 + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) tr[R1 * k2] = v[k2];
      }
    }
  }
}

// P1 (N grid): column IFFT_N -> p_N; I - |p_N|^2; column FFT_N -> T rows of Q
__device__ __noinline__ void ph_cols_rhs_n(const Args& a, const Ctx& c, int slot, int tile, unsigned g, unsigned G) {
  const DarkDev& L = *c.Lp();
  const int line = int(threadIdx.x) & 15, tt = int(threadIdx.x) >> 4;
  const size_t ii = size_t(tile) * a.t.n_img + a.t.nb + L.led;
  __syncthreads();
  for (int st = g; st < N / 16; st += G) {
    const int x = st * 16 + line;
    float2* tc = a.T + size_t(slot) * (N * N) + x;
    float2 v[16];
    float im[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int fy = tt + 16 * r, ky = fy < N / 2 ? fy : fy - N;
      v[r] = unsigned(ky - L.d_row0) < unsigned(L.d_nrow) ? __ldcg(&tc[fy * N]) : make_float2(0.f, 0.f);
      im[r] = img_load(a.src, ii, N * N, fy * N + x);
    }
    fft_regs<N, true, true>(v, c.bufA() + line * S256::LS, tt, c.tw256());
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = make_float2(im[r] - (v[r].x * v[r].x + v[r].y * v[r].y), 0.f);   // Eq. 13 lhs, spatial
    fft_regs<N, false, true>(v, c.bufA() + line * S256::LS, tt, c.tw256());
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int fy = tt + 16 * r, ky = fy < N / 2 ? fy : fy - N;
      if (unsigned(ky - L.q_row0) < unsigned(L.q_nrow)) tc[fy * N] = v[r];
    }
  }
}

// P1' (reduced grid): TM columns (rows of the disc) -> column IFFT_my -> p_M
template <int R1>
__device__ __noinline__ void ph_cols_pm(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  using M = XY<R1, true>;
  const DarkDev& L = *c.Lp();
  constexpr int my = 16 * R1;
  const int mx = L.mx, n_st = mx >> 4, d0 = modp(L.d_row0, my);
  const float2* tm = a.TM + size_t(slot) * (N * N);
  float2* pf = a.PF + size_t(slot) * (N * N);
  int par = 0;
  __syncthreads();
  for (int st = g; st < n_st; st += G, par ^= 1) {
    const int x = st * 16 + M::a_line(), t = M::a_t();
    float2 v[16];
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      v[r] = row_in(gy, d0, L.d_nrow, my) ? __ldcg(&tm[gy * mx + x]) : make_float2(0.f, 0.f);
    }
    fft_x<R1, true, true>(v, par ? c.bufB() : c.bufA(), c.twy());
    if (M::b_active()) {
      float2* pc = pf + M::b_k1() * mx + x;
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) pc[(R1 * k2) * mx] = v[k2];
    }
  }
}

// P2' : T rows of Q (N grid): row FFT_N, M_Q / N^2 = d on Q (Eq. 13), moved to the reduced grid, row IFFT_mx -> TM
template <int R1>
__device__ __noinline__ void ph_rows_rhs(const Args& a, const Ctx& c, int slot, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.q_nrow + 15) >> 4;
  const int line = int(threadIdx.x) >> 4, tt = int(threadIdx.x) & 15;
  const float scale = 1.f / float(N * N);
  const float2* tb = a.T + size_t(slot) * (N * N);
  float2* tm = a.TM + size_t(slot) * (N * N);
  __syncthreads();
  for (int st = g; st < n_st; st += G) {
    const int row = st * 16 + line;
    const bool valid = row < L.q_nrow;
    const int fy = wrapN(L.q_row0 + row);
    float2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = valid ? __ldcg(&tb[fy * N + tt + 16 * r]) : make_float2(0.f, 0.f);
    fft_regs<N, false, true>(v, c.bufB() + line * S256::LS, tt, c.tw256());
    // bin kx = tt + 16 r (r < 8) or tt + 16 (r - 16) (r >= 8) goes to reduced-grid column kx mod mx = tt + 16 r'
    float2 w[16];
#pragma unroll
    for (int r = 0; r < R1; ++r) w[r] = make_float2(0.f, 0.f);
    const int32_t* qrow = L.qmap + fy * L.q_ncol;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int rb = r < 8 ? r : r - 16;
      const int cc = tt + 16 * rb - L.q_col0;
      const int rp = ((rb % R1) + R1) % R1;
      if (valid && unsigned(cc) < unsigned(L.q_ncol) && __ldg(&qrow[cc]) >= 0) w[rp] = cadd(w[rp], cscale(v[r], scale));
    }
    fft_x<R1, true, false>(w, c.bufA(), c.twx());
    if (M::b_active()) {
      const int rowb = st * 16 + M::b_line(), k1 = M::b_k1();
      if (rowb < L.q_nrow) {
        float2* tr = tm + modp(L.q_row0 + rowb, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) tr[R1 * k2] = w[k2];
      }
    }
  }
}

// ================================================================ CG vector steps (redundant per CTA)
__device__ __forceinline__ float cg_init(const Args& a, const Ctx& c, int slot, int n_unknown) {
  const float2* wv = a.vec_w + size_t(slot) * a.max_unknown;
  float gsum = 0.f;
  for (int e = threadIdx.x; e < n_unknown; e += TH) {
    const float2 s = __ldcg(&wv[e]);
    c.ss()[e] = s;
    c.ps()[e] = s;
    c.xs()[e] = make_float2(0.f, 0.f);
    gsum += s.x * s.x + s.y * s.y;
  }
  return block_sum(gsum, c.red());
}
// Returns true when converged (||C^H r|| <= tol ||C^H d||) or when no progress is possible.
__device__ __forceinline__ bool cg_update(const Args& a, const Ctx& c, int slot, int n_unknown, float& gamma, float gamma0) {
  const float2* wv = a.vec_w + size_t(slot) * a.max_unknown;
  constexpr int PER = 8;                               // entries per thread held in registers (<= 2048 unknowns)
  float2 wr[PER];
  float pw = 0.f;
#pragma unroll
  for (int i = 0; i < PER; ++i) {
    const int e = threadIdx.x + i * TH;
    if (e < n_unknown) {
      wr[i] = __ldcg(&wv[e]);
      const float2 p = c.ps()[e];
      pw += p.x * wr[i].x + p.y * wr[i].y;             // Re(conj(pdir) w) = ||C pdir||^2
    }
  }
  for (int e = threadIdx.x + PER * TH; e < n_unknown; e += TH) {
    const float2 w = __ldcg(&wv[e]), p = c.ps()[e];
    pw += p.x * w.x + p.y * w.y;
  }
  pw = block_sum(pw, c.red());
  if (!(pw > 0.f)) return true;
  const float alpha = gamma / pw;
  float gsum = 0.f;
#pragma unroll
  for (int i = 0; i < PER; ++i) {
    const int e = threadIdx.x + i * TH;
    if (e < n_unknown) {
      const float2 p = c.ps()[e];
      float2 x = c.xs()[e], s = c.ss()[e];
      x.x += alpha * p.x; x.y += alpha * p.y;
      s.x -= alpha * wr[i].x; s.y -= alpha * wr[i].y;
      c.xs()[e] = x;
      c.ss()[e] = s;
      gsum += s.x * s.x + s.y * s.y;
    }
  }
  for (int e = threadIdx.x + PER * TH; e < n_unknown; e += TH) {
    const float2 w = __ldcg(&wv[e]), p = c.ps()[e];
    float2 x = c.xs()[e], s = c.ss()[e];
    x.x += alpha * p.x; x.y += alpha * p.y;
    s.x -= alpha * w.x; s.y -= alpha * w.y;
    c.xs()[e] = x;
    c.ss()[e] = s;
    gsum += s.x * s.x + s.y * s.y;
  }
  gsum = block_sum(gsum, c.red());
  const float beta = gsum / gamma;
  for (int e = threadIdx.x; e < n_unknown; e += TH) {
    const float2 s = c.ss()[e], p = c.ps()[e];
    c.ps()[e] = make_float2(s.x + beta * p.x, s.y + beta * p.y);
  }
  gamma = gsum;
  return !(gsum > a.tol2 * gamma0);
}

}  // namespace mg

// ================================================================ the kernel
__global__ void __launch_bounds__(mg::TH, 2) df_mgrid_kernel(const __grid_constant__ mg::Args a) {
  using namespace mg;
  Ctx c;
  c.mu = a.max_unknown;
  float2* tws = c.twx();                               // [3][256]: rows, columns, N grid
  float* c_sh = c.c_sh();
  DarkDev& Lsh = *c.Lp();
  const unsigned G = cluster_size(), g = cluster_rank();
  const bool multi = G > 1;
  const int team_id = blockIdx.x / G, n_teams = gridDim.x / G;
  tws[512 + threadIdx.x] = a.t.tw_xy[4 * 256 + threadIdx.x];
  const int live_n = *a.live_count - a.chunk0;
  const int tiles = live_n < a.n_tiles ? live_n : a.n_tiles;
  const int nz = a.t.nz;
  double flop = 0.0;
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
      const int r1x = Lsh.mx >> 4, r1y = Lsh.my >> 4;
      tws[threadIdx.x] = a.t.tw_xy[tw_slot(r1x) * 256 + threadIdx.x];
      tws[256 + threadIdx.x] = a.t.tw_xy[tw_slot(r1y) * 256 + threadIdx.x];
      __syncthreads();
      const int n_d = (Lsh.d_nrow + 15) >> 4, n_q = (Lsh.q_nrow + 15) >> 4, n_u = (Lsh.u_nrow + 15) >> 4, n_c = Lsh.mx >> 4;
      const double fx = 16.0 * line_flop(Lsh.mx), fy = 16.0 * line_flop(Lsh.my), fn = 16.0 * line_flop(N);
      // ---- setup: P_hat -> p_N, p_M -> d on Q -> s = C^H d
      ph_build_p_rows_n(a, c, slot, g, G);
      with_r1(r1x, [&](auto R) { ph_build_p_rows_m<decltype(R)::value>(a, c, slot, g, G); });
      team_sync(multi);
      ph_cols_rhs_n(a, c, slot, tile, g, G);
      with_r1(r1y, [&](auto R) { ph_cols_pm<decltype(R)::value>(a, c, slot, g, G); });
      team_sync(multi);
      with_r1(r1x, [&](auto R) { ph_rows_rhs<decltype(R)::value>(a, c, slot, g, G); });
      team_sync(multi);
      with_r1(r1y, [&](auto R) { ph_cols_mul<decltype(R)::value, false>(a, c, slot, g, G); });
      team_sync(multi);
      with_r1(r1x, [&](auto R) { ph_rows_u_gather<decltype(R)::value>(a, c, slot, g, G); });
      team_sync(multi);
      flop += mine(n_d) * (fn + fx) + mine(N / 16) * 2 * fn + mine(n_c) * fy + mine(n_q) * (fn + fx) + mine(n_c) * 2 * fy +
              mine(n_u) * fx;
      float gamma = cg_init(a, c, slot, n_unknown);
      const float gamma0 = gamma;
      int iters = 0;
      bool done = !(gamma > 0.f);
      // ---- CG on the normal equations
      while (!done && iters < a.max_iters) {
        __syncthreads();                                   // pdir complete in shared memory
        with_r1(r1x, [&](auto R) { ph_rows_u_scatter<decltype(R)::value>(a, c, slot, g, G); });
        team_sync(multi);
        with_r1(r1y, [&](auto R) { ph_cols_mul<decltype(R)::value, true>(a, c, slot, g, G); });
        team_sync(multi);
        with_r1(r1x, [&](auto R) { ph_rows_q<decltype(R)::value>(a, c, slot, g, G); });
        team_sync(multi);
        with_r1(r1y, [&](auto R) { ph_cols_mul<decltype(R)::value, false>(a, c, slot, g, G); });
        team_sync(multi);
        with_r1(r1x, [&](auto R) { ph_rows_u_gather<decltype(R)::value>(a, c, slot, g, G); });
        team_sync(multi);
        flop += 2 * mine(n_u) * fx + 4 * mine(n_c) * fy + 2 * mine(n_q) * fx;
        done = cg_update(a, c, slot, n_unknown, gamma, gamma0);
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
          const float2 u = cmulc(c.xs()[e], make_float2(cs, sn));
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
  if (threadIdx.x == 0 && flop > 0.0) atomicAdd(a.work, (unsigned long long)(flop + 0.5));
}

void launch_darkfield_mgrid(const DevTables& t, const DarkDev* d_leds, int n_leds, const Workspace& w, const LaunchCtx& c,
                            const ImgSrc& src, int df_iters, float df_tol, int team_size) {
  using namespace mg;
  if (n_leds <= 0) return;
  const size_t smem = (size_t(kSmFixed) + 3 * size_t(w.max_unknown)) * sizeof(float2);
  const int sms = c.pd->sms;
  if (!c.pd->attr_mgrid) {
    cudaFuncSetAttribute(df_mgrid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 4096);
    cudaFuncSetAttribute(df_mgrid_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    c.pd->attr_mgrid = true;
  }
  Args a{};
  a.t = t; a.leds = d_leds; a.n_leds = n_leds; a.src = src; a.O = w.O; a.coef = w.coef; a.T = w.T; a.TM = w.TM;
  a.PF = w.PF; a.vec_w = w.vec_w; a.cg_iters = w.cg_iters; a.max_unknown = w.max_unknown; a.max_iters = df_iters;
  a.tol2 = df_tol * df_tol; a.live = c.live; a.live_count = c.live_count; a.chunk0 = c.chunk0;
  a.n_tiles = c.chunk_tiles; a.work = w.df_work;
  int G = team_size;
  if (G <= 0) {
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, df_mgrid_kernel, TH, smem);
    per_sm = std::max(1, per_sm);
    // as many CTAs per tile as the pass leaves resident slots for.  Measured on config 2 (ms per step): 32 tiles
    // G = 8: 8.3; 56 tiles G = 5: 10.4; 64 tiles G = 4: 12.1; cluster sizes 6 and 7 place badly (40 tiles G = 7: 15.7,
    // 48 tiles G = 6: 16.3) and are skipped.
    G = 1;
    for (int cand : {8, 5, 4, 2})
      if (cand * c.chunk_tiles <= sms * per_sm) { G = cand; break; }
  }
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = unsigned(G); at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeClusterSchedulingPolicyPreference;
  at[1].val.clusterSchedulingPolicyPreference = cudaClusterSchedulingPolicyLoadBalancing;   // measured: 10.35 vs 10.58 ms (default / spread)
  cfg.blockDim = dim3(TH);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = c.stream;
  cfg.attrs = at;
  cfg.numAttrs = 2;
  int max_clusters = 0;
  cfg.gridDim = dim3(unsigned(G) * unsigned(sms / G));
  if (cudaOccupancyMaxActiveClusters(&max_clusters, df_mgrid_kernel, &cfg) != cudaSuccess || max_clusters < 1)
    max_clusters = std::max(1, sms / G - (G > 2 ? 2 : 0));
  const int teams = std::max(1, std::min(max_clusters, c.chunk_tiles));
  cfg.gridDim = dim3(unsigned(G) * unsigned(teams));
  ProfScope ps(c, CAT_DF_MGRID);
  cudaLaunchKernelEx(&cfg, df_mgrid_kernel, a);
}

// ================================================================ apic_fft2d_xy (kernel-level parity tests)
namespace mg {
// one pass over the rows (COLS = false) or columns (COLS = true) of [batch][my][mx]; mode as in apic.h
template <int R1, bool COLS>
__global__ void __launch_bounds__(TH) xy_pass_kernel(float2* d, int mx, int my, int mode, const float2* tw_xy) {
  using M = XY<R1, COLS>;
  __shared__ float2 bufA[kXyBuf];
  float2* bufB = bufA;
  __shared__ float2 tw[256];
  tw[threadIdx.x] = tw_xy[tw_slot(R1) * 256 + threadIdx.x];
  __syncthreads();
  float2* img = d + size_t(blockIdx.y) * mx * my;
  const int st = blockIdx.x;
  const int stride = COLS ? mx : 1, lstride = COLS ? 1 : mx;
  const int n_lines = COLS ? mx : my;
  float2 v[16];
  {
    const int ln = st * 16 + M::a_line(), t = M::a_t();
#pragma unroll
    for (int r = 0; r < R1; ++r) v[r] = ln < n_lines ? img[size_t(ln) * lstride + size_t(t + 16 * r) * stride] : make_float2(0.f, 0.f);
  }
  const bool inv = (mode == 1 || mode == 2);
  if (inv) fft_x<R1, true, COLS>(v, bufA, tw); else fft_x<R1, false, COLS>(v, bufA, tw);
  if (mode < 2) {
    if (M::b_active()) {
      const int ln = st * 16 + M::b_line(), k1 = M::b_k1();
      if (ln < n_lines) {
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) img[size_t(ln) * lstride + size_t(k1 + R1 * k2) * stride] = v[k2];
      }
    }
    return;
  }
  const float sc = 1.f / float(16 * R1);
#pragma unroll
  for (int k2 = 0; k2 < 16; ++k2) v[k2] = cscale(v[k2], sc);
  __syncthreads();                                      // single exchange buffer here
  if (inv) fft_y<R1, false, COLS>(v, bufB, tw); else fft_y<R1, true, COLS>(v, bufB, tw);
  {
    const int ln = st * 16 + M::a_line(), t = M::a_t();
    if (ln < n_lines) {
#pragma unroll
      for (int r = 0; r < R1; ++r) img[size_t(ln) * lstride + size_t(t + 16 * r) * stride] = v[r];
    }
  }
}
template <bool COLS>
void xy_pass(float2* d, int mx, int my, int batch, int mode, const float2* tw, cudaStream_t s) {
  const int len = COLS ? my : mx, lines = COLS ? mx : my;
  dim3 grid((lines + 15) / 16, batch);
  switch (len / 16) {
    case 6: xy_pass_kernel<6, COLS><<<grid, TH, 0, s>>>(d, mx, my, mode, tw); break;
    case 8: xy_pass_kernel<8, COLS><<<grid, TH, 0, s>>>(d, mx, my, mode, tw); break;
    case 10: xy_pass_kernel<10, COLS><<<grid, TH, 0, s>>>(d, mx, my, mode, tw); break;
    case 12: xy_pass_kernel<12, COLS><<<grid, TH, 0, s>>>(d, mx, my, mode, tw); break;
    default: xy_pass_kernel<16, COLS><<<grid, TH, 0, s>>>(d, mx, my, mode, tw); break;
  }
}
}  // namespace mg

int launch_fft2d_xy(float2* d, int mx, int my, int batch, int mode, const float2* tw_xy, cudaStream_t s) {
  mg::xy_pass<false>(d, mx, my, batch, mode, tw_xy, s);
  mg::xy_pass<true>(d, mx, my, batch, mode, tw_xy, s);
  return 0;
}

}  // namespace apic
