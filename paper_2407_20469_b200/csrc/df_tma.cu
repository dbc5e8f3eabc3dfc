// df_tma.cu - S8-S10 darkfield extension on per-LED reduced cyclic grids with async-proxy (TMA bulk copy) staging
// (df_mode 4 at N = 256; df_mgrid.cu is the same solver with plain loads, df_mode 0).
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
// Scheduling: one launch per pass covers every LED; a thread-block cluster (team) owns a tile, its
// CTAs split the 16-line strips of each phase and meet at cluster barriers.  Line transforms are
// fft_xy.cuh's X/Y pair.
//
// Data movement.  The reduced-grid scratch TM and p_M are stored STRIP-MAJOR,
//     idx(x, y) = (x / 16) * (16 my) + y * 16 + (x % 16),
// so that a column strip (16 columns x my rows) is ONE contiguous block and a row strip (16 rows x mx
// columns) is mx/16 contiguous 2 KB blocks.  Strips are staged into shared memory by the async proxy
// (cp.async.bulk global -> shared, completion on an mbarrier; SASS: UBLKCP.S.G / SYNCS.*): the last warp
// issues the copies of the next strips while the CTA transforms the current one, p_M strips (static per
// LED) are requested before the cluster barrier that precedes their phase, and the transform threads
// read their operands from shared memory without address arithmetic and without holding p in registers.
// Results are stored from registers (coalesced 128-byte segments); every thread executes
// fence.proxy.async before the cluster barrier (release / acquire), which orders those generic-proxy
// stores before the next phase's bulk loads.
// Measured on config 2 (profiles/r2_darkfield.md): the staging removes the operand waits of all but the
// first strip of a phase, but a strip is bound by the dependent-instruction latency of its two register
// transforms at 16 resident warps per SM, and the first strip of a phase pays the bulk copy's latency
// after the barrier: 11.2 ms per 64-tile launch against 10.4 ms for df_mgrid.cu's plain loads, so this
// kernel is the explicitly named alternative (df_mode 4), not the default.
//
// The CG vectors x, s, pdir, w are DISTRIBUTED: a CTA keeps only the entries of the U-row strips it
// transforms in phases A / E (U entries are row-major, so a strip's entries are one contiguous range).
// The dot products of an iteration, <pdir, w>, <s, w>, <w, w> and <s, s>, are reduced together: every
// CTA writes its four partial sums into every team member's shared memory (DSMEM) before the cluster
// barrier that ends phase E, and all members add them in the same order, so alpha, beta and the
// convergence decision are bit-identical across the team.  ||s_new||^2 = ||s||^2 - 2 alpha <s, w> +
// alpha^2 <w, w> gives beta without a second reduction; ||s||^2 itself is recomputed directly in the
// next iteration's reduction, so the recurrence never accumulates error.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <type_traits>
#include <vector>

#include "fft_xy.cuh"
#include "plan.hpp"

namespace apic {
namespace tma {

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
  float2* X;               // [chunk][max_unknown] CG iterate
  int max_unknown;
  int32_t* cg_iters;
  int kbuf;                // float2 entries of one staging / exchange buffer in shared memory
  int kpbuf;               // float2 entries of the p_M strip buffer
  int cap_local;           // capacity of a CTA's share of the CG vectors (entries)
  int max_iters;
  float tol2;
  const int32_t* live;
  const int32_t* live_count;
  int chunk0, n_tiles;
  unsigned long long* work;   // executed nominal flop (5 L log2 L per line transform)
};
#ifdef APIC_TIMELINE
constexpr int kTlCap = 4096;
__device__ unsigned long long* g_tl_dbg = nullptr;
// clock64 mark of thread 0 of the CTAs of team 0; the write index lives in shared memory (misc float 250)
#define TL_MARK(id)                                                                                          \
  do {                                                                                                       \
    if (g_tl_dbg && blockIdx.x < cluster_size() && threadIdx.x == 0) {                                       \
      unsigned* n_ = reinterpret_cast<unsigned*>(c.misc() + 250);                                            \
      if (*n_ + 1 < kTlCap) {                                                                                \
        g_tl_dbg[size_t(cluster_rank()) * kTlCap + *n_ + 1] = (unsigned long long)(clock64() << 8) | unsigned(id); \
        g_tl_dbg[size_t(cluster_rank()) * kTlCap] = ++*n_;                                                   \
      }                                                                                                      \
    }                                                                                                        \
  } while (0)
#else
#define TL_MARK(id) do {} while (0)
#endif

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
// Every thread orders its generic-proxy global stores before later async-proxy (bulk copy) reads of the team.
__device__ __forceinline__ void team_sync(bool multi) {
  asm volatile("fence.proxy.async;" ::: "memory");
  if (multi) {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
  } else {
    __syncthreads();
  }
}
// ---- async proxy: bulk copies global -> shared completing on an mbarrier (SASS: UBLKCP / SYNCS)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return uint32_t(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// strip-major index of grid point (x, y) on an mx x my grid
__device__ __forceinline__ int sm_idx(int x, int y, int my) { return (x >> 4) * (my << 4) + (y << 4) + (x & 15); }
__device__ __forceinline__ int wrapm(int k, int m) { return k >= m ? k - m : k; }   // k mod m for k in [0, 2m)
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

// R1_SWITCH(r1, call using R): the call with the compile-time constant R = r1 (arguments stay in registers)
#define R1_SWITCH(r1, ...)                                    \
  switch (r1) {                                               \
    case 6: { constexpr int R = 6; __VA_ARGS__; } break;      \
    case 8: { constexpr int R = 8; __VA_ARGS__; } break;      \
    case 10: { constexpr int R = 10; __VA_ARGS__; } break;    \
    case 12: { constexpr int R = 12; __VA_ARGS__; } break;    \
    default: { constexpr int R = 16; __VA_ARGS__; } break;    \
  }

// Shared-memory layout of a CTA (all dynamic, float2 units; kb = Args::kbuf, kp = Args::kpbuf, cap = Args::cap_local):
//   [L0 kb][L1 kb][EY kb][PB kp][twx 256][twy 256][tw256 256][misc 128][ss cap][ps cap]
// L0 / L1: landing buffers of the bulk copies (a strip of TM), reused as the X-exchange buffer of the strip they held;
//          together they hold the 16 x 273 strip of the N-grid transforms of the set-up phases.
// EY: Y-exchange buffer; between phase E and the vector update it holds w (this CTA's share; cap <= kb).
// The iterate x is only touched by the vector update (each entry by one fixed thread) and lives in global memory
// (Args::X), which leaves a few KB of the SM's shared memory / L1 carve-out to the L1 cache.
// PB: landing buffer of a p_M column strip (16 columns x my rows).
// misc (floats): [0,64) Zernike coefficients of the tile, [64,96) reduction scratch, [96,128) the team's partial dot
//          products [8][4], [128,134) three mbarriers (L0, L1, PB), [136,184) the current DarkDev.
struct Ctx {
  int kb, kp, cap;
  __device__ __forceinline__ float2* base() const {
    extern __shared__ __align__(128) float2 dyn[];
    return dyn;
  }
  __device__ __forceinline__ float2* land(int i) const { return base() + i * kb; }
  __device__ __forceinline__ float2* ey() const { return base() + 2 * kb; }
  __device__ __forceinline__ float2* pb() const { return base() + 3 * kb; }
  __device__ __forceinline__ float2* twx() const { return base() + 3 * kb + kp; }
  __device__ __forceinline__ float2* twy() const { return twx() + 256; }
  __device__ __forceinline__ float2* tw256() const { return twx() + 512; }
  __device__ __forceinline__ float* misc() const { return reinterpret_cast<float*>(twx() + 768); }
  __device__ __forceinline__ float* c_sh() const { return misc(); }
  __device__ __forceinline__ float* red() const { return misc() + 64; }
  __device__ __forceinline__ float4* slots() const { return reinterpret_cast<float4*>(misc() + 96); }
  __device__ __forceinline__ uint64_t* mbar() const { return reinterpret_cast<uint64_t*>(misc() + 128); }
  __device__ __forceinline__ DarkDev* Lp() const { return reinterpret_cast<DarkDev*>(misc() + 136); }
  __device__ __forceinline__ float2* ss() const { return twx() + 768 + 128; }
  __device__ __forceinline__ float2* ps() const { return ss() + cap; }
  __device__ __forceinline__ float2* ws() const { return ey(); }
};
constexpr int kSmFixed = 768 + 128;                 // float2 entries besides the four buffers and the CG vectors
constexpr int kMinBuf = 2192;                       // 2 kb >= 16 x 273 (S256 strip of the set-up phases)
constexpr int kMaxTeam = 8;
static_assert(sizeof(DarkDev) <= (256 - 136) * sizeof(float), "DarkDev does not fit the misc region");
static_assert(sizeof(DarkDev) % sizeof(int) == 0, "DarkDev is copied as ints");
static_assert(kMaxZern <= 64, "c_sh region");
static_assert(2 * kMinBuf >= 16 * S256::LS, "N-grid strip buffer");
enum { BAR_L0 = 0, BAR_L1 = 1, BAR_P = 2 };

constexpr int kIssue = TH - 32;   // the last warp issues the bulk copies: in the layout-B stages it has no transform work (R1 < 16)
// ---- staging (the last warp issues; `par` holds the phase parity of each mbarrier, uniform across the CTA)
// column strip: rows [in0, in0 + in_n) (mod my) of one strip-major column strip -> buf[row * 16 + col]
__device__ __forceinline__ void issue_cols(const Ctx& c, int which, const float2* strip, int in0, int in_n, int my) {
  if (threadIdx.x >= kIssue) {
    const int lane = int(threadIdx.x) - kIssue;
    const int n1 = min(in_n, my - in0), n2 = in_n - n1;
    uint64_t* bar = c.mbar() + which;
    if (lane == 0) mbar_expect_tx(bar, unsigned(in_n) * 128u);
    __syncwarp();
    if (lane == 0) bulk_g2s(c.land(which) + in0 * 16, strip + in0 * 16, unsigned(n1) * 128u, bar);
    if (lane == 1 && n2 > 0) bulk_g2s(c.land(which), strip, unsigned(n2) * 128u, bar);
  }
}
// row strip: nv rows starting at physical row pr0 (wrapping at my), pieces r < r1x -> buf[r * 256 + line * 16 + t]
__device__ __forceinline__ void issue_rows(const Ctx& c, int which, const float2* tm, int pr0, int nv, int my, int r1x) {
  if (threadIdx.x >= kIssue) {
    const int lane = int(threadIdx.x) - kIssue;
    const int n1 = min(nv, my - pr0), n2 = nv - n1;
    uint64_t* bar = c.mbar() + which;
    if (lane == 0) mbar_expect_tx(bar, unsigned(nv * r1x) * 128u);
    __syncwarp();
    if (lane < r1x) {
      const float2* src = tm + lane * (my << 4);
      float2* dst = c.land(which) + lane * 256;
      bulk_g2s(dst, src + pr0 * 16, unsigned(n1) * 128u, bar);
      if (n2 > 0) bulk_g2s(dst + n1 * 16, src, unsigned(n2) * 128u, bar);
    }
  }
}
__device__ __forceinline__ void land_wait(const Ctx& c, int which, unsigned& par) {
  mbar_wait(c.mbar() + which, (par >> which) & 1u);
  par ^= 1u << which;
}
// p_M column strip `st` of this tile -> PB.  Every thread of the CTA must be past its last read of PB.
__device__ __forceinline__ void prefetch_p(const Ctx& c, const float2* pf, int st) {
  const DarkDev& L = *c.Lp();
  if (threadIdx.x == kIssue && st < (L.mx >> 4)) {
    const unsigned bytes = unsigned(L.my) * 128u;
    mbar_expect_tx(c.mbar() + BAR_P, bytes);
    bulk_g2s(c.pb(), pf + size_t(st) * (L.my << 4), bytes, c.mbar() + BAR_P);
  }
}

// ================================================================ reduced-grid phases
// A: E_U pdir (this CTA's share, shared memory) -> row IFFT_mx -> TM rows of U
template <int R1>
__device__ __noinline__ void ph_rows_u_scatter(const Ctx c, float2* tm, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.u_nrow + 15) >> 4;
  int par = 0, lb = 0;
  for (int st = g; st < n_st; st += G, par ^= 1) {
    const int e0 = L.u_strip_off[st], e1 = L.u_strip_off[st + 1];
    float2 v[16];
    {
      const int row = st * 16 + M::a_line(), t = M::a_t();
      const int32_t* drow = L.dmap_m + wrapm(L.u0m + row, my) * mx;
#pragma unroll
      for (int r = 0; r < R1; ++r) {
        v[r] = make_float2(0.f, 0.f);
        if (row < L.u_nrow) {
          const int e = __ldg(&drow[t + 16 * r]);
          if (unsigned(e - e0) < unsigned(e1 - e0)) v[r] = c.ps()[lb + e - e0];
        }
      }
    }
    fft_x<R1, true, false>(v, c.land(par), c.twx());
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.u_nrow) {
        float2* tr = tm + (wrapm(L.u0m + row, my) << 4);
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const int x = k1 + R1 * k2;
          tr[(x >> 4) * (my << 4) + (x & 15)] = v[k2];
        }
      }
    }
    lb += e1 - e0;
  }
}

// E: TM rows of U -> row FFT_mx -> gather U -> w / (mx my) (this CTA's share, shared memory)
template <int R1>
__device__ __noinline__ unsigned ph_rows_u_gather(const Ctx c, const float2* tm, unsigned g, unsigned G, unsigned par) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.u_nrow + 15) >> 4;
  const float scale = 1.f / float(mx * my);
  const int u0 = L.u0m;
  for (int j = 0; j < 2; ++j) {
    const int st = int(g) + j * int(G);
    if (st < n_st) issue_rows(c, j, tm, wrapm(u0 + st * 16, my), min(16, L.u_nrow - st * 16), my, R1);
  }
  int i = 0, lb = 0;
  for (int st = g; st < n_st; st += G, ++i) {
    const int e0 = L.u_strip_off[st], e1 = L.u_strip_off[st + 1];
    float2* lbuf = c.land(i & 1);
    float2 v[16];
    land_wait(c, i & 1, par);
    {
      const int line = M::a_line(), t = M::a_t();
      const bool valid = st * 16 + line < L.u_nrow;
#pragma unroll
      for (int r = 0; r < R1; ++r) v[r] = valid ? lbuf[r * 256 + line * 16 + t] : make_float2(0.f, 0.f);
    }
    __syncthreads();                                    // landing data in registers: the buffer becomes the exchange
    fft_x<R1, false, false>(v, lbuf, c.twx());
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.u_nrow) {
        const int32_t* drow = L.dmap_m + wrapm(L.u0m + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const int e = __ldg(&drow[R1 * k2]);
          if (unsigned(e - e0) < unsigned(e1 - e0)) c.ws()[lb + e - e0] = cscale(v[k2], scale);
        }
      }
    }
    lb += e1 - e0;
    if (st + 2 * int(G) < n_st) {
      __syncthreads();                                  // every thread is past its exchange reads
      issue_rows(c, i & 1, tm, wrapm(u0 + (st + 2 * int(G)) * 16, my), min(16, L.u_nrow - (st + 2 * int(G)) * 16), my, R1);
    }
  }
  return par;
}

// C: TM rows of Q: row FFT_mx, M_Q / (mx my), row IFFT_mx
template <int R1>
__device__ __noinline__ unsigned ph_rows_q(const Ctx c, float2* tm, unsigned g, unsigned G, unsigned par) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.q_nrow + 15) >> 4;
  const float scale = 1.f / float(mx * my);
  const int q0 = L.q0m;
  for (int j = 0; j < 2; ++j) {
    const int st = int(g) + j * int(G);
    if (st < n_st) issue_rows(c, j, tm, wrapm(q0 + st * 16, my), min(16, L.q_nrow - st * 16), my, R1);
  }
  int i = 0;
  for (int st = g; st < n_st; st += G, ++i) {
    float2* lbuf = c.land(i & 1);
    float2 v[16];
    const int line = M::a_line(), t = M::a_t();
    const bool valid = st * 16 + line < L.q_nrow;
    unsigned keep = 0;
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.q_nrow) {
        const uint8_t* qrow = L.qmask_m + wrapm(q0 + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) keep |= unsigned(__ldg(&qrow[R1 * k2]) != 0) << k2;
      }
    }
    land_wait(c, i & 1, par);
#pragma unroll
    for (int r = 0; r < R1; ++r) v[r] = valid ? lbuf[r * 256 + line * 16 + t] : make_float2(0.f, 0.f);
    __syncthreads();
    fft_x<R1, false, false>(v, lbuf, c.twx());
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) v[k2] = (keep >> k2 & 1u) ? cscale(v[k2], scale) : make_float2(0.f, 0.f);
    fft_y<R1, true, false>(v, c.ey(), c.twx());
    if (st + 2 * int(G) < n_st)                         // fft_y's barrier: every thread is past its reads of lbuf
      issue_rows(c, i & 1, tm, wrapm(q0 + (st + 2 * int(G)) * 16, my), min(16, L.q_nrow - (st + 2 * int(G)) * 16), my, R1);
    if (valid) {
      float2* tr = tm + (wrapm(q0 + st * 16 + line, my) << 4) + t;
#pragma unroll
      for (int r = 0; r < R1; ++r) tr[r * (my << 4)] = v[r];
    }
  }
  return par;
}

// B / D: TM columns: IFFT_my, . conj p_M (B) or . p_M (D), FFT_my.  The p_M strip of the CTA's first column strip
// has been requested by prefetch_p before the cluster barrier that precedes the phase.
template <int R1, bool CONJ>
__device__ __noinline__ unsigned ph_cols_mul(const Ctx c, float2* tm, const float2* pf, unsigned g, unsigned G, unsigned par) {
  using M = XY<R1, true>;
  const DarkDev& L = *c.Lp();
  constexpr int my = 16 * R1;
  const int mx = L.mx, n_st = mx >> 4;
  const int in0 = CONJ ? L.u0m : L.q0m, in_n = CONJ ? L.u_nrow : L.q_nrow;
  const int out0 = CONJ ? L.q0m : L.u0m, out_n = CONJ ? L.q_nrow : L.u_nrow;
  for (int j = 0; j < 2; ++j) {
    const int st = int(g) + j * int(G);
    if (st < n_st) issue_cols(c, j, tm + size_t(st) * (16 * my), in0, in_n, my);
  }
  int i = 0;
  for (int st = g; st < n_st; st += G, ++i) {
    float2* lbuf = c.land(i & 1);
    float2* strip = tm + size_t(st) * (16 * my);
    const int line = M::a_line(), t = M::a_t();
    float2 v[16];
    TL_MARK(20);
    land_wait(c, i & 1, par);
    TL_MARK(21);
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      v[r] = row_in(gy, in0, in_n, my) ? lbuf[gy * 16 + line] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    TL_MARK(22);
    fft_x<R1, true, true>(v, lbuf, c.twy());
    TL_MARK(23);
    land_wait(c, BAR_P, par);
    TL_MARK(24);
    if (M::b_active()) {
      const float2* pc = c.pb() + M::b_k1() * 16 + line;
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) {
        const float2 p = pc[(R1 * k2) * 16];
        v[k2] = CONJ ? cmulc(v[k2], p) : cmul(v[k2], p);
      }
    }
    fft_y<R1, false, true>(v, c.ey(), c.twy());
    TL_MARK(25);
    // fft_y's barrier: every thread is past its reads of lbuf and PB
    prefetch_p(c, pf, st + int(G));
    if (st + 2 * int(G) < n_st) issue_cols(c, i & 1, tm + size_t(st + 2 * int(G)) * (16 * my), in0, in_n, my);
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      if (row_in(gy, out0, out_n, my)) strip[gy * 16 + line] = v[r];
    }
    TL_MARK(26);
  }
  return par;
}

// ================================================================ setup phases
__device__ __forceinline__ int wrapN(int k) { return (k + N) & (N - 1); }
__device__ __forceinline__ float2 p_hat_entry(const Ctx& c, const float2* __restrict__ o, int e, int nz) {
  // P_hat(k) = O_hat(k) e^{+j phi(k + kappa)} on P = D_i ∩ known
  const DarkDev& L = *c.Lp();
  const float phi = zern_phase(L.zern + size_t(e) * nz, c.c_sh(), nz);
  float sn, cs;
  sincosf(phi, &sn, &cs);
  return cmul(__ldcg(&o[__ldg(&L.disc_f[e])]), make_float2(cs, sn));
}

// P0 (N grid): P_hat rows -> row IFFT_N -> T
__device__ __noinline__ void ph_build_p_rows_n(const Ctx c, const float2* o, float2* tn, int nz, unsigned g, unsigned G) {
  const DarkDev& L = *c.Lp();
  const int line = int(threadIdx.x) >> 4, tt = int(threadIdx.x) & 15;
  const int n_st = (L.d_nrow + 15) >> 4;
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
        if (e >= L.n_unknown) v[r] = p_hat_entry(c, o, e, nz);
      }
    }
    fft_regs<N, true, true>(v, c.land(0) + line * S256::LS, tt, c.tw256());
    if (valid) {
      float2* tr = tn + fy * N;
#pragma unroll
      for (int r = 0; r < 16; ++r) tr[tt + 16 * r] = v[r];
    }
  }
}

// P0' (reduced grid): P_hat rows -> row IFFT_mx -> TM
template <int R1>
__device__ __noinline__ void ph_build_p_rows_m(const Ctx c, const float2* o, float2* tm, int nz, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.d_nrow + 15) >> 4;
  int par = 0;
  __syncthreads();                                     // L0 / L1 held the strip of the N-grid transform
  for (int st = g; st < n_st; st += G, par ^= 1) {
    float2 v[16];
    {
      const int row = st * 16 + M::a_line(), t = M::a_t();
      const int32_t* drow = L.dmap_m + wrapm(L.d0m + row, my) * mx;
#pragma unroll
      for (int r = 0; r < R1; ++r) {
        v[r] = make_float2(0.f, 0.f);
        if (row < L.d_nrow) {
          const int e = __ldg(&drow[t + 16 * r]);
          if (e >= L.n_unknown) v[r] = p_hat_entry(c, o, e, nz);
        }
      }
    }
    fft_x<R1, true, false>(v, c.land(par), c.twx());
    if (M::b_active()) {
      const int row = st * 16 + M::b_line(), k1 = M::b_k1();
      if (row < L.d_nrow) {
        float2* tr = tm + (wrapm(L.d0m + row, my) << 4);
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const int x = k1 + R1 * k2;
          tr[(x >> 4) * (my << 4) + (x & 15)] = v[k2];
        }
      }
    }
  }
}

// P1 (N grid): column IFFT_N -> p_N; I - |p_N|^2; column FFT_N -> T rows of Q
__device__ __noinline__ void ph_cols_rhs_n(const Ctx c, float2* tn, const ImgSrc src, size_t ii, unsigned g, unsigned G) {
  const DarkDev& L = *c.Lp();
  const int line = int(threadIdx.x) & 15, tt = int(threadIdx.x) >> 4;
  __syncthreads();
  for (int st = g; st < N / 16; st += G) {
    const int x = st * 16 + line;
    float2* tc = tn + x;
    float2 v[16];
    float im[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int fy = tt + 16 * r, ky = fy < N / 2 ? fy : fy - N;
      v[r] = unsigned(ky - L.d_row0) < unsigned(L.d_nrow) ? __ldcg(&tc[fy * N]) : make_float2(0.f, 0.f);
      im[r] = img_load(src, ii, N * N, fy * N + x);
    }
    fft_regs<N, true, true>(v, c.land(0) + line * S256::LS, tt, c.tw256());
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = make_float2(im[r] - (v[r].x * v[r].x + v[r].y * v[r].y), 0.f);   // Eq. 13 lhs, spatial
    fft_regs<N, false, true>(v, c.land(0) + line * S256::LS, tt, c.tw256());
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int fy = tt + 16 * r, ky = fy < N / 2 ? fy : fy - N;
      if (unsigned(ky - L.q_row0) < unsigned(L.q_nrow)) tc[fy * N] = v[r];
    }
  }
}

// P1' (reduced grid): TM columns (rows of the disc) -> column IFFT_my -> p_M (strip-major, like TM)
template <int R1>
__device__ __noinline__ void ph_cols_pm(const Ctx c, const float2* tm, float2* pf, unsigned g, unsigned G) {
  using M = XY<R1, true>;
  const DarkDev& L = *c.Lp();
  constexpr int my = 16 * R1;
  const int mx = L.mx, n_st = mx >> 4, d0 = L.d0m;
  int par = 0;
  __syncthreads();
  for (int st = g; st < n_st; st += G, par ^= 1) {
    const int line = M::a_line(), t = M::a_t();
    const float2* strip = tm + size_t(st) * (16 * my);
    float2 v[16];
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      v[r] = row_in(gy, d0, L.d_nrow, my) ? __ldcg(&strip[gy * 16 + line]) : make_float2(0.f, 0.f);
    }
    fft_x<R1, true, true>(v, par ? c.pb() : c.ey(), c.twy());
    if (M::b_active()) {
      float2* pc = pf + size_t(st) * (16 * my) + M::b_k1() * 16 + line;
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) pc[(R1 * k2) * 16] = v[k2];
    }
  }
}

// P2' : T rows of Q (N grid): row FFT_N, M_Q / N^2 = d on Q (Eq. 13), moved to the reduced grid, row IFFT_mx -> TM
template <int R1>
__device__ __noinline__ void ph_rows_rhs(const Ctx c, const float2* tb, float2* tm, unsigned g, unsigned G) {
  using M = XY<R1, false>;
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.q_nrow + 15) >> 4;
  const int line = int(threadIdx.x) >> 4, tt = int(threadIdx.x) & 15;
  const float scale = 1.f / float(N * N);
  __syncthreads();
  for (int st = g; st < n_st; st += G) {
    const int row = st * 16 + line;
    const bool valid = row < L.q_nrow;
    const int fy = wrapN(L.q_row0 + row);
    float2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = valid ? __ldcg(&tb[fy * N + tt + 16 * r]) : make_float2(0.f, 0.f);
    fft_regs<N, false, true>(v, c.land(0) + line * S256::LS, tt, c.tw256());
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
    fft_x<R1, true, false>(w, c.ey(), c.twx());
    if (M::b_active()) {
      const int rowb = st * 16 + M::b_line(), k1 = M::b_k1();
      if (rowb < L.q_nrow) {
        float2* tr = tm + (wrapm(L.q0m + rowb, my) << 4);
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const int x = k1 + R1 * k2;
          tr[(x >> 4) * (my << 4) + (x & 15)] = w[k2];
        }
      }
    }
  }
}

// ================================================================ CG vector steps (each CTA on its share)
// Partial sums of this CTA's entries -> every team member's slot [g] (DSMEM).  init: s = pdir = w, x = 0 first.
__device__ __forceinline__ void cg_partials(const Ctx& c, int n_own, bool init, unsigned g, unsigned G) {
  __syncthreads();                                      // w of phase E complete in shared memory
  float pw = 0.f, sw = 0.f, ww = 0.f, s2 = 0.f;
  for (int j = threadIdx.x; j < n_own; j += TH) {
    const float2 w = c.ws()[j];
    if (init) {
      c.ss()[j] = w;
      c.ps()[j] = w;
      s2 += w.x * w.x + w.y * w.y;
    } else {
      const float2 p = c.ps()[j], s = c.ss()[j];
      pw += p.x * w.x + p.y * w.y;                      // Re(conj(pdir) w) = ||C pdir||^2
      sw += s.x * w.x + s.y * w.y;
      ww += w.x * w.x + w.y * w.y;
      s2 += s.x * s.x + s.y * s.y;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    pw += __shfl_xor_sync(0xffffffffu, pw, o);
    sw += __shfl_xor_sync(0xffffffffu, sw, o);
    ww += __shfl_xor_sync(0xffffffffu, ww, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
  }
  float4* red = reinterpret_cast<float4*>(c.red());
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = make_float4(pw, sw, ww, s2);
  __syncthreads();
  if (threadIdx.x < G) {
    float4 s = red[0];
#pragma unroll
    for (int i = 1; i < TH / 32; ++i) {
      const float4 q = red[i];
      s.x += q.x; s.y += q.y; s.z += q.z; s.w += q.w;
    }
    unsigned remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(c.slots() + g)), "r"(unsigned(threadIdx.x)));
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(remote), "f"(s.x), "f"(s.y), "f"(s.z), "f"(s.w) : "memory");
  }
}
__device__ __forceinline__ float4 cg_totals(const Ctx& c, unsigned G) {   // after the team barrier
  float4 s = c.slots()[0];
  for (unsigned q = 1; q < G; ++q) {
    const float4 r = c.slots()[q];
    s.x += r.x; s.y += r.y; s.z += r.z; s.w += r.w;
  }
  return s;
}
// x += alpha pdir (global memory, entry e of the LED's unknowns; first = the iterate starts from 0), s -= alpha w,
// pdir = s + beta pdir.  Entry (strip st, j) is always handled by thread j mod TH of the CTA that owns the strip.
__device__ __forceinline__ void cg_update(const Ctx& c, float2* __restrict__ xg, unsigned g, unsigned G, float alpha, float beta,
                                          bool first) {
  const DarkDev& L = *c.Lp();
  const int n_u = (L.u_nrow + 15) >> 4;
  int lb = 0;
  for (int st = g; st < n_u; st += G) {
    const int e0 = L.u_strip_off[st], cnt = L.u_strip_off[st + 1] - e0;
    for (int j = threadIdx.x; j < cnt; j += TH) {
      const float2 p = c.ps()[lb + j], w = c.ws()[lb + j];
      float2 x = first ? make_float2(0.f, 0.f) : __ldcg(&xg[e0 + j]), s = c.ss()[lb + j];
      x.x += alpha * p.x; x.y += alpha * p.y;
      s.x -= alpha * w.x; s.y -= alpha * w.y;
      xg[e0 + j] = x;
      c.ss()[lb + j] = s;
      c.ps()[lb + j] = make_float2(s.x + beta * p.x, s.y + beta * p.y);
    }
    lb += cnt;
  }
}

}  // namespace tma

// ================================================================ the kernel
__global__ void __launch_bounds__(tma::TH, 2) df_tma_kernel(const __grid_constant__ tma::Args a) {
  using namespace tma;
  Ctx c;
  c.kb = a.kbuf;
  c.kp = a.kpbuf;
  c.cap = a.cap_local;
  float2* tws = c.twx();                               // [3][256]: rows, columns, N grid
  float* c_sh = c.c_sh();
  DarkDev& Lsh = *c.Lp();
  const unsigned G = cluster_size(), g = cluster_rank();
  const bool multi = G > 1;
  const int team_id = blockIdx.x / G, n_teams = gridDim.x / G;
  if (threadIdx.x == 0) {
    mbar_init(c.mbar() + BAR_L0, 1);
    mbar_init(c.mbar() + BAR_L1, 1);
    mbar_init(c.mbar() + BAR_P, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  tws[512 + threadIdx.x] = a.t.tw_xy[4 * 256 + threadIdx.x];
#ifdef APIC_TIMELINE
  if (threadIdx.x == 0) *reinterpret_cast<unsigned*>(c.misc() + 250) = 0;
#endif
  __syncthreads();
  unsigned par = 0;                                     // phase parity of the three mbarriers
  const int live_n = *a.live_count - a.chunk0;
  const int tiles = live_n < a.n_tiles ? live_n : a.n_tiles;
  const int nz = a.t.nz;
  double flop = 0.0;
  auto mine = [&](int n_st) { return (n_st > int(g)) ? (n_st - int(g) + int(G) - 1) / int(G) : 0; };

  for (int slot = team_id; slot < tiles; slot += n_teams) {
    const int tile = a.live[a.chunk0 + slot];
    float2* const o_t = a.O + size_t(slot) * (N * N);   // this tile's object spectrum and scratch grids
    float2* const tn_t = a.T + size_t(slot) * (N * N);
    float2* const tm_t = a.TM + size_t(slot) * (N * N);
    float2* const pf_t = a.PF + size_t(slot) * (N * N);
    float2* const xg_t = a.X + size_t(slot) * a.max_unknown;
    __syncthreads();
    if (threadIdx.x < nz) c_sh[threadIdx.x] = a.coef[size_t(slot) * nz + threadIdx.x];
    for (int k = 0; k < a.n_leds; ++k) {
      __syncthreads();
      if (threadIdx.x < sizeof(DarkDev) / sizeof(int))
        reinterpret_cast<int*>(&Lsh)[threadIdx.x] = reinterpret_cast<const int*>(&a.leds[k])[threadIdx.x];
      __syncthreads();
      const int r1x = Lsh.mx >> 4, r1y = Lsh.my >> 4;
      tws[threadIdx.x] = a.t.tw_xy[tw_slot(r1x) * 256 + threadIdx.x];
      tws[256 + threadIdx.x] = a.t.tw_xy[tw_slot(r1y) * 256 + threadIdx.x];
      __syncthreads();
      const int n_d = (Lsh.d_nrow + 15) >> 4, n_q = (Lsh.q_nrow + 15) >> 4, n_u = (Lsh.u_nrow + 15) >> 4, n_c = Lsh.mx >> 4;
      const double fx = 16.0 * line_flop(Lsh.mx), fy = 16.0 * line_flop(Lsh.my), fn = 16.0 * line_flop(N);
      TL_MARK(100 + k);
      int n_own = 0;                                     // this CTA's share of the unknowns: its U-row strips
      for (int st = g; st < n_u; st += G) n_own += Lsh.u_strip_off[st + 1] - Lsh.u_strip_off[st];
      // ---- setup: P_hat -> p_N, p_M -> d on Q -> s = C^H d
      ph_build_p_rows_n(c, o_t, tn_t, nz, g, G);
      R1_SWITCH(r1x, ph_build_p_rows_m<R>(c, o_t, tm_t, nz, g, G));
      team_sync(multi);
      ph_cols_rhs_n(c, tn_t, a.src, size_t(tile) * a.t.n_img + a.t.nb + Lsh.led, g, G);
      R1_SWITCH(r1y, ph_cols_pm<R>(c, tm_t, pf_t, g, G));
      team_sync(multi);
      R1_SWITCH(r1x, ph_rows_rhs<R>(c, tn_t, tm_t, g, G));
      prefetch_p(c, pf_t, int(g));
      team_sync(multi);
      R1_SWITCH(r1y, par = ph_cols_mul<R, false>(c, tm_t, pf_t, g, G, par));
      team_sync(multi);
      R1_SWITCH(r1x, par = ph_rows_u_gather<R>(c, tm_t, g, G, par));
      cg_partials(c, n_own, true, g, G);
      team_sync(multi);
      flop += mine(n_d) * (fn + fx) + mine(N / 16) * 2 * fn + mine(n_c) * fy + mine(n_q) * (fn + fx) + mine(n_c) * 2 * fy +
              mine(n_u) * fx;
      TL_MARK(12);
      const float gamma0 = cg_totals(c, G).w;
      int iters = 0;
      bool done = !(gamma0 > 0.f), have_x = false;
      // ---- CG on the normal equations
      while (!done && iters < a.max_iters) {
        __syncthreads();                                   // pdir complete in shared memory
        TL_MARK(1);
        R1_SWITCH(r1x, ph_rows_u_scatter<R>(c, tm_t, g, G));
        prefetch_p(c, pf_t, int(g));
        TL_MARK(2);
        team_sync(multi);
        TL_MARK(3);
        R1_SWITCH(r1y, par = ph_cols_mul<R, true>(c, tm_t, pf_t, g, G, par));
        TL_MARK(4);
        team_sync(multi);
        TL_MARK(5);
        R1_SWITCH(r1x, par = ph_rows_q<R>(c, tm_t, g, G, par));
        prefetch_p(c, pf_t, int(g));
        TL_MARK(6);
        team_sync(multi);
        TL_MARK(7);
        R1_SWITCH(r1y, par = ph_cols_mul<R, false>(c, tm_t, pf_t, g, G, par));
        TL_MARK(8);
        team_sync(multi);
        TL_MARK(9);
        R1_SWITCH(r1x, par = ph_rows_u_gather<R>(c, tm_t, g, G, par));
        cg_partials(c, n_own, false, g, G);
        TL_MARK(10);
        team_sync(multi);
        TL_MARK(11);
        flop += 2 * mine(n_u) * fx + 4 * mine(n_c) * fy + 2 * mine(n_q) * fx;
        ++iters;
        const float4 tot = cg_totals(c, G);                // <pdir, w>, <s, w>, <w, w>, <s, s>
        if (!(tot.x > 0.f)) break;
        const float gamma = tot.w, alpha = gamma / tot.x;
        const float gnew = fmaxf(gamma - 2.f * alpha * tot.y + alpha * alpha * tot.z, 0.f);   // ||s - alpha w||^2
        cg_update(c, xg_t, g, G, alpha, gnew / gamma, !have_x);
        have_x = true;
        done = !(gnew > a.tol2 * gamma0);
      }
      __syncthreads();
      // ---- S10: O_hat(u) = U_hat(u) e^{-j phi(u+kappa)}, known ∪= U (every CTA extends with its share)
      {
        float2* o = o_t;
        int lb = 0;
        for (int st = g; st < n_u; st += G) {
          const int e0 = Lsh.u_strip_off[st], cnt = Lsh.u_strip_off[st + 1] - e0;
          for (int j = threadIdx.x; j < cnt; j += TH) {
            const int e = e0 + j;
            const float phi = zern_phase(Lsh.zern + size_t(e) * nz, c_sh, nz);
            float sn, cs;
            sincosf(phi, &sn, &cs);
            const float2 x = have_x ? __ldcg(&xg_t[e]) : make_float2(0.f, 0.f);
            const int q = Lsh.disc_f[e];
            const float2 u = cmulc(x, make_float2(cs, sn));
            o[q] = Lsh.accumulate ? cadd(__ldcg(&o[q]), u) : u;   // ring-wise order (R15b): sum now, mean at the end of the ring
          }
          lb += cnt;
        }
        if (g == 0 && threadIdx.x == 0) a.cg_iters[size_t(slot) * a.n_leds + k] = iters;
      }
      team_sync(multi);                                    // O complete before the next LED reads it
      if (Lsh.n_avg > 0) {                                 // df_order 1, end of a ring: bins solved by c LEDs hold a sum of c solutions
        float2* o = o_t;
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

void launch_darkfield_tma(const DevTables& t, const DarkDev* d_leds, const DarkDev* h_leds, int n_leds, const Workspace& w,
                            const LaunchCtx& c, const ImgSrc& src, int df_iters, float df_tol, int team_size) {
  using namespace tma;
  if (n_leds <= 0) return;
  const int sms = c.pd->sms;
  if (!c.pd->attr_tma) {
    cudaFuncSetAttribute(df_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
    cudaFuncSetAttribute(df_tma_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    c.pd->attr_tma = true;
  }
  // staging / exchange buffers sized by the largest line of any LED's grid (16 lines x R1 x 18 padded entries)
  int r1max = 6;
  for (int k = 0; k < n_leds; ++k) r1max = std::max(r1max, std::max(h_leds[k].mx, h_leds[k].my) >> 4);
  const int kb0 = std::max(kMinBuf, 16 * r1max * 18), kp = 256 * r1max;
  // a CTA's share of the CG vectors: the entries of the U-row strips g, g + G, ... (largest over LEDs and members)
  auto cap_for = [&](int G) {
    int cap = 2;
    for (int k = 0; k < n_leds; ++k) {
      const int n_u = (h_leds[k].u_nrow + 15) >> 4;
      for (int g = 0; g < G; ++g) {
        int s = 0;
        for (int st = g; st < n_u; st += G) s += h_leds[k].u_strip_off[st + 1] - h_leds[k].u_strip_off[st];
        cap = std::max(cap, s);
      }
    }
    return (cap + 1) & ~1;
  };
  const int kb = std::max(kb0, cap_for(1));             // w (a CTA's share) is kept in the Y-exchange buffer
  auto smem_for = [&](int G) { return (size_t(3 * kb + kp + kSmFixed) + 2 * size_t(cap_for(G))) * sizeof(float2); };
  int G = std::min(team_size, kMaxTeam);
  if (G <= 0) {
    // as many CTAs per tile as the pass leaves resident slots for (cluster sizes 6 and 7 place badly and are skipped)
    G = 1;
    for (int cand : {8, 5, 4, 2}) {
      int per_sm = 0;
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, df_tma_kernel, TH, smem_for(cand));
      if (per_sm >= 1 && cand * c.chunk_tiles <= sms * per_sm) { G = cand; break; }
    }
  }
  Args a{};
  a.t = t; a.leds = d_leds; a.n_leds = n_leds; a.src = src; a.O = w.O; a.coef = w.coef; a.T = w.T; a.TM = w.TM;
  a.PF = w.PF; a.X = w.vec_x; a.max_unknown = w.max_unknown; a.cg_iters = w.cg_iters; a.kbuf = kb; a.kpbuf = kp; a.cap_local = cap_for(G); a.max_iters = df_iters;
  a.tol2 = df_tol * df_tol; a.live = c.live; a.live_count = c.live_count; a.chunk0 = c.chunk0;
  a.n_tiles = c.chunk_tiles; a.work = w.df_work;
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = unsigned(G); at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeClusterSchedulingPolicyPreference;
  at[1].val.clusterSchedulingPolicyPreference = cudaClusterSchedulingPolicyLoadBalancing;
  cfg.blockDim = dim3(TH);
  cfg.dynamicSmemBytes = smem_for(G);
  cfg.stream = c.stream;
  cfg.attrs = at;
  cfg.numAttrs = 2;
  int max_clusters = 0;
  cfg.gridDim = dim3(unsigned(G) * unsigned(sms / G));
  if (cudaOccupancyMaxActiveClusters(&max_clusters, df_tma_kernel, &cfg) != cudaSuccess || max_clusters < 1)
    max_clusters = std::max(1, sms / G - (G > 2 ? 2 : 0));
  const int teams = std::max(1, std::min(max_clusters, c.chunk_tiles));
  cfg.gridDim = dim3(unsigned(G) * unsigned(teams));
#ifdef APIC_TIMELINE
  // debugging aid (build with -DAPIC_TIMELINE): APIC_DF_TIMELINE=<file> dumps the clock64 marks of team 0
#if defined(APIC_DF_KNOBS) || defined(APIC_TIMELINE)
  static const char* const tl_env = getenv("APIC_DF_TIMELINE");
#else
  static constexpr const char* tl_env = nullptr;        // the shipped library reads no environment variable
#endif
  const char* tl_path = tl_env;
  unsigned long long* dbg = nullptr;
  if (tl_path) {
    cudaMalloc(&dbg, size_t(kMaxTeam) * kTlCap * sizeof(unsigned long long));
    cudaMemsetAsync(dbg, 0, size_t(kMaxTeam) * kTlCap * sizeof(unsigned long long), c.stream);
  }
  cudaMemcpyToSymbolAsync(g_tl_dbg, &dbg, sizeof(dbg), 0, cudaMemcpyHostToDevice, c.stream);
#endif
  {
    ProfScope ps(c, CAT_DF_TMA);
    cudaLaunchKernelEx(&cfg, df_tma_kernel, a);
  }
#ifdef APIC_TIMELINE
  if (tl_path) {
    std::vector<unsigned long long> h(size_t(kMaxTeam) * kTlCap);
    cudaStreamSynchronize(c.stream);
    cudaMemcpy(h.data(), dbg, h.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    cudaFree(dbg);
    if (FILE* f = fopen(tl_path, "w")) {
      for (int q = 0; q < G; ++q)
        for (unsigned long long i = 1; i <= h[size_t(q) * kTlCap]; ++i)
          fprintf(f, "%d %llu %llu\n", q, h[size_t(q) * kTlCap + i] >> 8, h[size_t(q) * kTlCap + i] & 255ull);
      fclose(f);
    }
  }
#endif
}

}  // namespace apic
