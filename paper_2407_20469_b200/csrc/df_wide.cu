// df_wide.cu - S8-S10 darkfield extension on per-LED reduced cyclic grids, "wide" scheduling: the default darkfield kernel at N = 256
// (df_mode 0: 256-thread CTAs at 128 registers; df_mode 5: its 1024-thread shape, a measured alternative).
//
// Same mathematics as df_mgrid.cu (Eq. 11-13; readings R15-R17, B1): per darkfield LED, conjugate
// gradients on the normal equations of  C u = d,  C[k,u] = conj P_hat(u - k), k in Q, u in U, with C and C^H applied by
// FFTs on the LED's alias-free reduced cyclic grid mx x my (geometry.cpp); only the right-hand side
// d = F(I - |p|^2)/N^2 (Eq. 13) runs on the N x N grid, once per LED.
//
// What differs is how a tile's chain of phases is scheduled.  df_mgrid.cu runs 2 CTAs of 256 threads per SM at 128
// registers: 16 warps per SM, and a phase of 6-10 strips takes 2-3 sequential strip rounds on a team of 4 CTAs.  The
// step time there is the length of the per-tile dependency chain (profiles/r1b_cfg2_mgrid.md), so here
//   * a CTA holds NG GROUPS of 256 threads (NG = 4: 1024 threads, one CTA per SM; NG = 2: 512 threads, two per SM), every
//     thread is compiled for 64 registers, and each group transforms its own 16-line strip with its own exchange buffer
//     and its own named barrier (bar.sync id, 256): a team of G CTAs offers S = G NG strip SLOTS per tile (8 for G = 2),
//     so most phases are ONE strip round and an SM keeps 32 warps in flight;
//   * nothing that is static across the CG iterations of a LED is fetched twice: a slot's p_M column strip (the
//     pointwise factor of phases B / D) is parked in shared memory by the very threads that multiply with it
//     (thread-private, so no barrier), and the Q mask bits of a slot's row strip live in one shared-memory word per thread;
//     p is never held in registers across a transform (that is what kept df_mgrid.cu at 128 registers);
//   * the CG vectors x, s, pdir, w are DISTRIBUTED over the slots: a slot keeps the entries of the U-row strips it
//     transforms in phases A / E (U entries are row-major, so a strip's entries are one contiguous range).  The dot
//     products of an iteration, <pdir, w>, <s, w>, <w, w>, <s, s>, are reduced together: the owner of a 16-row strip of U
//     writes the strip's four partial sums into every team member's shared memory (DSMEM) before the cluster barrier
//     that ends phase E and all threads add the strips' sums in strip order, so alpha, beta and the convergence decision
//     are bit-identical across the team AND independent of the team size (a batch gives the same bits however it is
//     split into passes).  ||s_new||^2 = ||s||^2 - 2 alpha <s, w> + alpha^2 <w, w> gives beta without a second reduction;
//     ||s||^2 itself is recomputed directly in the next iteration's reduction, so the recurrence never accumulates error.
// The scratch grids TM / PF stay row-major in L2 as in df_mgrid.cu; the line transforms are fft_xy.cuh's X / Y pair and
// fft_core.cuh's radix-16 pair with a group-local barrier.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <vector>

#include "fft_xy.cuh"
#include "plan.hpp"

namespace apic {
namespace wd {

constexpr int N = 256;
constexpr int GT = 256;      // threads of a group = one 16-line strip
using S256 = Strip<256>;     // N-grid line transform of fft_core.cuh (16 lines x 16 threads)
constexpr int kMaxSlots = 16;

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
  float2* VW;              // [chunk][max_unknown] w, s, x of the CG when they do not fit shared memory (vec_global bits)
  float2* VS;
  float2* VX;
  int max_unknown;
  int vec_global;          // bit 0: w in global memory, bit 1: s, bit 2: x (pdir always lives in shared memory)
  int vr;                  // 1: LEDs that fit run the decimated CG loop (pairs of 1024-thread CTAs)
  int vr_mu;               // capacity of each of the four redundant CG vectors of that loop (entries)
  int32_t* cg_iters;
  int kex;                 // float2 entries of a group's exchange buffer
  int kpc;                 // float2 entries of a group's p_M strip cache (directly behind the exchange buffer)
  int cap;                 // capacity of a slot's share of the CG vectors (entries)
  int max_iters;
  float tol2;
  const int32_t* live;
  const int32_t* live_count;
  int chunk0, n_tiles;
  unsigned long long* work;   // executed nominal flop (5 L log2 L per line transform)
  unsigned long long* tl;     // optional timeline of team 0 (-DAPIC_DF_KNOBS builds: APIC_DF_TIMELINE=<file>): [cta][group][kTlCap] clock marks
};
constexpr int kTlCap = 8192;
#ifdef APIC_TIMELINE   // debugging aid: build with APIC_EXTRA_NVCC_FLAGS=-DAPIC_TIMELINE, run with APIC_DF_TIMELINE=<file>
#define WD_MARK(id)                                                                                   \
  do {                                                                                                \
    if (a.tl && team_id == 0 && g.tid == 0 && tl_n + 1 < kTlCap) {                                    \
      unsigned long long t_;                                                                          \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                                          \
      a.tl[(size_t(cr) * NG + g.grp) * kTlCap + ++tl_n] = (t_ << 8) | unsigned(id);                   \
    }                                                                                                 \
  } while (0)
#else
#define WD_MARK(id) do {} while (0)
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
__device__ __forceinline__ void team_sync(bool multi) {
  if (multi) {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
  } else {
    __syncthreads();
  }
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return uint32_t(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ int wrapm(int k, int m) { return k >= m ? k - m : k; }   // k mod m for k in [0, 2m)
__device__ __forceinline__ int wrapN(int k) { return (k + N) & (N - 1); }
// is grid row g (0 <= g < m) one of the nrow rows starting at physical row row0m (mod m)?
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

// R1_SWITCH(r1, call using R): the call with the compile-time constant R = r1
#define WD_R1_SWITCH(r1, ...)                                 \
  switch (r1) {                                               \
    case 6: { constexpr int R = 6; __VA_ARGS__; } break;      \
    case 8: { constexpr int R = 8; __VA_ARGS__; } break;      \
    case 10: { constexpr int R = 10; __VA_ARGS__; } break;    \
    case 12: { constexpr int R = 12; __VA_ARGS__; } break;    \
    default: { constexpr int R = 16; __VA_ARGS__; } break;    \
  }

// A group of 256 threads inside the CTA and the strip slot it fills in the team.
struct Grp {
  int tid;      // 0..255 inside the group
  int grp;      // group index inside the CTA (named barrier 1 + grp)
  int sigma;    // slot in the team: strips sigma, sigma + S, ... of every phase
  int S;        // slots per team = cluster size x groups per CTA
};
__device__ __forceinline__ void gsync(const Grp& g) {
  asm volatile("bar.sync %0, %1;" ::"r"(g.grp + 1), "n"(GT) : "memory");
}

// Shared-memory layout of a CTA (all dynamic, float2 units; kex / kpc / cap from Args, NG groups):
//   [group 0: EX kex | PC kpc] ... [group NG-1: EX | PC] [twx 256][twy 256][tw256 256][misc 256][KQ NG x 128][CG NG x nvec x cap]
// EX: exchange buffer of the group's line transforms; EX and PC together hold the 16 x 273 strip of the N-grid
//     transforms of the set-up phases (PC is refilled afterwards).
// PC: p_M column strip of the slot's first strip of phases B / D, entry [k2][tid] written and read by the same thread.
// KQ: per thread, the 16 Q-mask bits of the slot's first row strip of phase C.
// CG: the slot's share of pdir and of those of w, s, x that fit (Args::vec_global).
// misc (floats): [0,64) Zernike coefficients of the tile, [64,128) the team's partial dot products [16][4],
//     [128,256) per-group reduction scratch [NG][8][4], [256,..) the current DarkDev.
struct Ctx {
  int kex, kpc, cap, ng, nvec;
  __device__ __forceinline__ float2* base() const {
    extern __shared__ __align__(16) float2 dyn[];
    return dyn;
  }
  __device__ __forceinline__ float2* ex(int grp) const { return base() + grp * (kex + kpc); }
  __device__ __forceinline__ float2* pc(int grp) const { return ex(grp) + kex; }
  __device__ __forceinline__ float2* twx() const { return base() + ng * (kex + kpc); }
  __device__ __forceinline__ float2* twy() const { return twx() + 256; }
  __device__ __forceinline__ float2* tw256() const { return twx() + 512; }
  __device__ __forceinline__ float* misc() const { return reinterpret_cast<float*>(twx() + 768); }
  __device__ __forceinline__ float* c_sh() const { return misc(); }
  __device__ __forceinline__ float4* totals() const { return reinterpret_cast<float4*>(misc() + 64); }
  __device__ __forceinline__ float4* red(int grp) const { return reinterpret_cast<float4*>(misc() + 128) + grp * 8; }
  __device__ __forceinline__ DarkDev* Lp() const { return reinterpret_cast<DarkDev*>(misc() + 256); }
  __device__ __forceinline__ unsigned* kq(int grp) const { return reinterpret_cast<unsigned*>(twx() + 768 + 256) + grp * 256; }
  __device__ __forceinline__ float2* cg(int grp) const { return twx() + 768 + 256 + ng * 128 + grp * nvec * cap; }
  __device__ __forceinline__ float2* ps(int grp) const { return cg(grp); }
};
// One of the CG vectors w, s, x of a slot: in the slot's shared memory (index = position in the slot's share) or in
// global memory (index = entry of the LED's unknowns), decided on the host from the shared-memory budget.
struct Vec {
  float2* p;
  int gl;
  __device__ __forceinline__ float2& operator()(int local, int entry) const { return p[gl ? entry : local]; }
};
struct Vecs { Vec w, s, x; };
static_assert(sizeof(DarkDev) <= 256 * sizeof(float), "DarkDev does not fit the misc region");
static_assert(sizeof(DarkDev) % sizeof(int) == 0, "DarkDev is copied as ints");
static_assert(kMaxZern <= 64, "c_sh region");
constexpr int kSmFixed = 768 + 256;   // float2 entries besides the per-group regions

// ================================================================ line transforms with a group-local barrier
// fft_xy.cuh's type X / type Y on ONE exchange buffer: the first barrier of each protects the buffer against the
// previous transform's readers (it comes after the register DFT, so it is rarely waited for).
template <int R1, bool INV, bool COLS>
__device__ __forceinline__ void fft_xg(float2 (&v)[16], const Grp& g, float2* __restrict__ buf, const float2* __restrict__ tw) {
  using M = XY<R1, COLS>;
  const int tid = g.tid;
  {
    float2 a[R1];
#pragma unroll
    for (int r = 0; r < R1; ++r) a[r] = v[r];
    RegDft<R1, INV>::run(a);
    const int line = COLS ? tid & 15 : tid >> 4, t = COLS ? tid >> 4 : tid & 15;
    gsync(g);
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) {
      const float2 y = k1 ? twmul<INV>(a[k1], tw[k1 * 16 + t]) : a[0];
      if (COLS) buf[(k1 * 16 + t) * 16 + line] = y;
      else buf[line * (R1 * 18) + k1 * 18 + t] = y;
    }
  }
  gsync(g);
  if (tid < 16 * R1) {
    const int line = COLS ? tid & 15 : tid / R1, k1 = COLS ? tid >> 4 : tid % R1;
    if (COLS) {
#pragma unroll
      for (int t = 0; t < 16; ++t) v[t] = buf[(k1 * 16 + t) * 16 + line];
    } else {
      const float4* src = reinterpret_cast<const float4*>(buf + line * (R1 * 18) + k1 * 18);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float4 q = src[i];
        v[2 * i] = make_float2(q.x, q.y);
        v[2 * i + 1] = make_float2(q.z, q.w);
      }
    }
    RegDft<16, INV>::run(v);
  }
}
template <int R1, bool INV, bool COLS>
__device__ __forceinline__ void fft_yg(float2 (&v)[16], const Grp& g, float2* __restrict__ buf, const float2* __restrict__ tw) {
  using M = XY<R1, COLS>;
  const int tid = g.tid;
  const bool act = tid < 16 * R1;
  if (act) RegDft<16, INV>::run(v);
  gsync(g);
  if (act) {
    const int line = COLS ? tid & 15 : tid / R1, k1 = COLS ? tid >> 4 : tid % R1;
#pragma unroll
    for (int kp = 0; kp < 16; ++kp) {
      const float2 y = kp ? twmul<INV>(v[kp], tw[kp * 16 + k1]) : v[0];
      if (COLS) buf[(kp * R1 + k1) * 16 + line] = y;
      else buf[line * M::LSY + kp * M::R1P + k1] = y;
    }
  }
  gsync(g);
  {
    const int line = COLS ? tid & 15 : tid >> 4, kp = COLS ? tid >> 4 : tid & 15;
    float2 a[R1];
    if (COLS) {
#pragma unroll
      for (int j = 0; j < R1; ++j) a[j] = buf[(kp * R1 + j) * 16 + line];
    } else {
      const float4* src = reinterpret_cast<const float4*>(buf + line * M::LSY + kp * M::R1P);
#pragma unroll
      for (int i = 0; i < R1 / 2; ++i) {
        const float4 q = src[i];
        a[2 * i] = make_float2(q.x, q.y);
        a[2 * i + 1] = make_float2(q.z, q.w);
      }
    }
    RegDft<R1, INV>::run(a);
#pragma unroll
    for (int r = 0; r < R1; ++r) v[r] = a[r];
  }
}
// fft_core.cuh's N = 256 line transform (radix 16 x 16): in v[r] = x[t + 16 r], out v[r] = X[t + 16 r]; `ln` = the
// thread's line in the group's strip buffer, `tw` = the 256-entry table in shared memory.
template <bool INV>
__device__ __forceinline__ void fft256g(float2 (&v)[16], const Grp& g, float2* __restrict__ ln, int t, const float2* __restrict__ tw) {
  RegDft<16, INV>::run(v);
#pragma unroll
  for (int k1 = 1; k1 < 16; ++k1) v[k1] = twmul<INV>(v[k1], tw[k1 * 16 + t]);
  gsync(g);
#pragma unroll
  for (int k1 = 0; k1 < 16; ++k1) ln[pad16(t + 16 * k1)] = v[k1];
  gsync(g);
#pragma unroll
  for (int n1 = 0; n1 < 16; ++n1) v[n1] = ln[pad16(16 * t + n1)];
  RegDft<16, INV>::run(v);
}

// ================================================================ reduced-grid phases
// A: E_U pdir (this slot's share, shared memory) -> row IFFT_mx -> TM rows of U
template <int R1>
__device__ __noinline__ void ph_rows_u_scatter(const Ctx c, const Grp g, float2* tm) {
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.u_nrow + 15) >> 4;
  const float2* ps = c.ps(g.grp);
  int lb = 0;
  for (int st = g.sigma; st < n_st; st += g.S) {
    const int e0 = L.u_strip_off[st], ne = L.u_strip_off[st + 1] - e0;
    float2 v[16];
    {
      const int row = st * 16 + (g.tid >> 4), t = g.tid & 15;
      const int32_t* drow = L.dmap_m + wrapm(L.u0m + row, my) * mx;
#pragma unroll
      for (int r = 0; r < R1; ++r) {
        v[r] = make_float2(0.f, 0.f);
        if (row < L.u_nrow) {
          const int e = __ldg(&drow[t + 16 * r]);
          if (unsigned(e - e0) < unsigned(ne)) v[r] = ps[lb + e - e0];
        }
      }
    }
    fft_xg<R1, true, false>(v, g, c.ex(g.grp), c.twx());
    if (g.tid < 16 * R1) {
      const int row = st * 16 + g.tid / R1, k1 = g.tid % R1;
      if (row < L.u_nrow) {
        float2* tr = tm + wrapm(L.u0m + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) tr[R1 * k2] = v[k2];
      }
    }
    lb += ne;
  }
}

// E: TM rows of U -> row FFT_mx -> gather U -> w / (mx my) (this slot's share, shared memory)
template <int R1>
__device__ __noinline__ void ph_rows_u_gather(const Ctx c, const Grp g, const float2* tm, const Vec vw) {
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.u_nrow + 15) >> 4;
  const float scale = 1.f / float(mx * my);
  int lb = 0;
  for (int st = g.sigma; st < n_st; st += g.S) {
    const int e0 = L.u_strip_off[st], ne = L.u_strip_off[st + 1] - e0;
    float2 v[16];
    {
      const int row = st * 16 + (g.tid >> 4), t = g.tid & 15;
      const float2* tr = tm + wrapm(L.u0m + row, my) * mx + t;
#pragma unroll
      for (int r = 0; r < R1; ++r) v[r] = row < L.u_nrow ? __ldcg(&tr[16 * r]) : make_float2(0.f, 0.f);
    }
    fft_xg<R1, false, false>(v, g, c.ex(g.grp), c.twx());
    if (g.tid < 16 * R1) {
      const int row = st * 16 + g.tid / R1, k1 = g.tid % R1;
      if (row < L.u_nrow) {
        const int32_t* drow = L.dmap_m + wrapm(L.u0m + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const int e = __ldg(&drow[R1 * k2]);
          if (unsigned(e - e0) < unsigned(ne)) vw(lb + e - e0, e) = cscale(v[k2], scale);
        }
      }
    }
    lb += ne;
  }
}

// Q-mask bits of the layout-B thread for row strip `st` (bit k2 <-> column k1 + R1 k2)
template <int R1>
__device__ __forceinline__ unsigned q_keep_bits(const DarkDev& L, int st, int tid) {
  constexpr int mx = 16 * R1;
  unsigned keep = 0;
  if (tid < 16 * R1) {
    const int row = st * 16 + tid / R1, k1 = tid % R1;
    if (row < L.q_nrow) {
      const uint8_t* qrow = L.qmask_m + wrapm(L.q0m + row, L.my) * mx + k1;
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) keep |= unsigned(__ldg(&qrow[R1 * k2]) != 0) << k2;
    }
  }
  return keep;
}

// C: TM rows of Q: row FFT_mx, M_Q / (mx my), row IFFT_mx
template <int R1>
__device__ __noinline__ void ph_rows_q(const Ctx c, const Grp g, float2* tm) {
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.q_nrow + 15) >> 4;
  const float scale = 1.f / float(mx * my);
  for (int st = g.sigma; st < n_st; st += g.S) {
    float2 v[16];
    const int rowa = st * 16 + (g.tid >> 4), t = g.tid & 15;
    float2* tr = tm + wrapm(L.q0m + rowa, my) * mx + t;
#pragma unroll
    for (int r = 0; r < R1; ++r) v[r] = rowa < L.q_nrow ? __ldcg(&tr[16 * r]) : make_float2(0.f, 0.f);
    fft_xg<R1, false, false>(v, g, c.ex(g.grp), c.twx());
    const unsigned keep = st == g.sigma ? c.kq(g.grp)[g.tid] : q_keep_bits<R1>(L, st, g.tid);
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) v[k2] = (keep >> k2 & 1u) ? cscale(v[k2], scale) : make_float2(0.f, 0.f);
    fft_yg<R1, true, false>(v, g, c.ex(g.grp), c.twx());
    if (rowa < L.q_nrow) {
#pragma unroll
      for (int r = 0; r < R1; ++r) tr[16 * r] = v[r];
    }
  }
}

// B / D: TM columns: IFFT_my, . conj p_M (B) or . p_M (D), FFT_my.  The p_M strip of the slot's first column strip is
// parked in PC by the threads that use it (fill = true: read it from PF and park it; false: read PC).
template <int R1, bool CONJ>
__device__ __noinline__ void ph_cols_mul(const Ctx c, const Grp g, float2* tm, const float2* pf, bool fill) {
  const DarkDev& L = *c.Lp();
  constexpr int my = 16 * R1;
  const int mx = L.mx, n_st = mx >> 4;
  const int in0 = CONJ ? L.u0m : L.q0m, in_n = CONJ ? L.u_nrow : L.q_nrow;
  const int out0 = CONJ ? L.q0m : L.u0m, out_n = CONJ ? L.q_nrow : L.u_nrow;
  const int line = g.tid & 15, t = g.tid >> 4;
  float2* pc = c.pc(g.grp) + g.tid;
  for (int st = g.sigma; st < n_st; st += g.S) {
    const int x = st * 16 + line;
    float2 v[16];
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      v[r] = row_in(gy, in0, in_n, my) ? __ldcg(&tm[gy * mx + x]) : make_float2(0.f, 0.f);
    }
    fft_xg<R1, true, true>(v, g, c.ex(g.grp), c.twy());
    if (t < R1) {
      if (st == g.sigma && !fill) {
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const float2 p = pc[k2 * (16 * R1)];
          v[k2] = CONJ ? cmulc(v[k2], p) : cmul(v[k2], p);
        }
      } else {
        const float2* pcol = pf + t * mx + x;
        const bool park = st == g.sigma;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
          const float2 p = __ldcg(&pcol[(R1 * k2) * mx]);
          if (park) pc[k2 * (16 * R1)] = p;
          v[k2] = CONJ ? cmulc(v[k2], p) : cmul(v[k2], p);
        }
      }
    }
    fft_yg<R1, false, true>(v, g, c.ex(g.grp), c.twy());
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      if (row_in(gy, out0, out_n, my)) tm[gy * mx + x] = v[r];
    }
  }
}

// ================================================================ setup phases
__device__ __forceinline__ float2 p_hat_entry(const Ctx& c, const float2* __restrict__ o, int e, int nz) {
  // P_hat(k) = O_hat(k) e^{+j phi(k + kappa)} on P = D_i ∩ known
  const DarkDev& L = *c.Lp();
  const float phi = zern_phase(L.zern + size_t(e) * nz, c.c_sh(), nz);
  float sn, cs;
  sincosf(phi, &sn, &cs);
  return cmul(__ldcg(&o[__ldg(&L.disc_f[e])]), make_float2(cs, sn));
}

// P0 (N grid): P_hat rows -> row IFFT_N -> T
__device__ __noinline__ void ph_build_p_rows_n(const Ctx c, const Grp g, const float2* o, float2* tn, int nz) {
  const DarkDev& L = *c.Lp();
  const int line = g.tid >> 4, tt = g.tid & 15;
  const int n_st = (L.d_nrow + 15) >> 4;
  for (int st = g.sigma; st < n_st; st += g.S) {
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
    fft256g<true>(v, g, c.ex(g.grp) + line * S256::LS, tt, c.tw256());
    if (valid) {
      float2* tr = tn + fy * N;
#pragma unroll
      for (int r = 0; r < 16; ++r) tr[tt + 16 * r] = v[r];
    }
  }
}

// P0' (reduced grid): P_hat rows -> row IFFT_mx -> TM
template <int R1>
__device__ __noinline__ void ph_build_p_rows_m(const Ctx c, const Grp g, const float2* o, float2* tm, int nz) {
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.d_nrow + 15) >> 4;
  for (int st = g.sigma; st < n_st; st += g.S) {
    float2 v[16];
    {
      const int row = st * 16 + (g.tid >> 4), t = g.tid & 15;
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
    fft_xg<R1, true, false>(v, g, c.ex(g.grp), c.twx());
    if (g.tid < 16 * R1) {
      const int row = st * 16 + g.tid / R1, k1 = g.tid % R1;
      if (row < L.d_nrow) {
        float2* tr = tm + wrapm(L.d0m + row, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) tr[R1 * k2] = v[k2];
      }
    }
  }
}

// P1 (N grid): column IFFT_N -> p_N; I - |p_N|^2; column FFT_N -> T rows of Q
__device__ __noinline__ void ph_cols_rhs_n(const Ctx c, const Grp g, float2* tn, const ImgSrc src, size_t ii) {
  const DarkDev& L = *c.Lp();
  const int line = g.tid & 15, tt = g.tid >> 4;
  for (int st = g.sigma; st < N / 16; st += g.S) {
    const int x = st * 16 + line;
    float2* tc = tn + x;
    float2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int fy = tt + 16 * r, ky = fy < N / 2 ? fy : fy - N;
      v[r] = unsigned(ky - L.d_row0) < unsigned(L.d_nrow) ? __ldcg(&tc[fy * N]) : make_float2(0.f, 0.f);
    }
    fft256g<true>(v, g, c.ex(g.grp) + line * S256::LS, tt, c.tw256());
#pragma unroll
    for (int r = 0; r < 16; ++r) {                       // Eq. 13 lhs, spatial
      const float im = img_load(src, ii, N * N, (tt + 16 * r) * N + x);
      v[r] = make_float2(im - (v[r].x * v[r].x + v[r].y * v[r].y), 0.f);
    }
    fft256g<false>(v, g, c.ex(g.grp) + line * S256::LS, tt, c.tw256());
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int fy = tt + 16 * r, ky = fy < N / 2 ? fy : fy - N;
      if (unsigned(ky - L.q_row0) < unsigned(L.q_nrow)) tc[fy * N] = v[r];
    }
  }
}

// P1' (reduced grid): TM columns (rows of the disc) -> column IFFT_my -> p_M
template <int R1>
__device__ __noinline__ void ph_cols_pm(const Ctx c, const Grp g, const float2* tm, float2* pf) {
  const DarkDev& L = *c.Lp();
  constexpr int my = 16 * R1;
  const int mx = L.mx, n_st = mx >> 4, d0 = L.d0m;
  const int line = g.tid & 15, t = g.tid >> 4;
  for (int st = g.sigma; st < n_st; st += g.S) {
    const int x = st * 16 + line;
    float2 v[16];
#pragma unroll
    for (int r = 0; r < R1; ++r) {
      const int gy = t + 16 * r;
      v[r] = row_in(gy, d0, L.d_nrow, my) ? __ldcg(&tm[gy * mx + x]) : make_float2(0.f, 0.f);
    }
    fft_xg<R1, true, true>(v, g, c.ex(g.grp), c.twy());
    if (t < R1) {
      float2* pcol = pf + t * mx + x;
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) pcol[(R1 * k2) * mx] = v[k2];
    }
  }
}

// P2' : T rows of Q (N grid): row FFT_N, M_Q / N^2 = d on Q (Eq. 13), moved to the reduced grid, row IFFT_mx -> TM
template <int R1>
__device__ __noinline__ void ph_rows_rhs(const Ctx c, const Grp g, const float2* tb, float2* tm) {
  const DarkDev& L = *c.Lp();
  constexpr int mx = 16 * R1;
  const int my = L.my, n_st = (L.q_nrow + 15) >> 4;
  const int line = g.tid >> 4, tt = g.tid & 15;
  const float scale = 1.f / float(N * N);
  for (int st = g.sigma; st < n_st; st += g.S) {
    const int row = st * 16 + line;
    const bool valid = row < L.q_nrow;
    const int fy = wrapN(L.q_row0 + row);
    float2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = valid ? __ldcg(&tb[fy * N + tt + 16 * r]) : make_float2(0.f, 0.f);
    fft256g<false>(v, g, c.ex(g.grp) + line * S256::LS, tt, c.tw256());
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
    fft_xg<R1, true, false>(w, g, c.ex(g.grp), c.twx());
    if (g.tid < 16 * R1) {
      const int rowb = st * 16 + g.tid / R1, k1 = g.tid % R1;
      if (rowb < L.q_nrow) {
        float2* tr = tm + wrapm(L.q0m + rowb, my) * mx + k1;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) tr[R1 * k2] = w[k2];
      }
    }
  }
}

// ================================================================ CG vector steps (each slot on its share)
// f(local, entry) for every entry of this slot's U-row strips
template <class F>
__device__ __forceinline__ void for_own(const DarkDev& L, const Grp& g, F&& f) {
  const int n_u = (L.u_nrow + 15) >> 4;
  int lb = 0;
  for (int st = g.sigma; st < n_u; st += g.S) {
    const int e0 = L.u_strip_off[st], cnt = L.u_strip_off[st + 1] - e0;
    for (int j = g.tid; j < cnt; j += GT) f(lb + j, e0 + j);
    lb += cnt;
  }
}
// Partial sums, one set per 16-row STRIP of U (not per slot, so that the association - and with it every bit of the
// result - does not depend on the team size or the groups per CTA): the slot that owns strip st reduces the strip's
// entries over its 256 threads in a fixed order and writes the four sums into totals[st] of every team member (DSMEM).
// init: s = pdir = w, x = 0 first.
__device__ __forceinline__ void cg_partials(const Ctx& c, const Grp& g, const Vecs& V, bool init, unsigned G) {
  const DarkDev& L = *c.Lp();
  const int n_u = (L.u_nrow + 15) >> 4;
  float2* ps = c.ps(g.grp);
  float4* red = c.red(g.grp);
  int lb = 0;
  gsync(g);                                             // w of phase E complete
  for (int st = g.sigma; st < n_u; st += g.S) {
    const int e0 = L.u_strip_off[st], cnt = L.u_strip_off[st + 1] - e0;
    float pw = 0.f, sw = 0.f, ww = 0.f, s2 = 0.f;
    for (int j = g.tid; j < cnt; j += GT) {
      const int l = lb + j, e = e0 + j;
      const float2 w = V.w(l, e);
      if (init) {
        V.s(l, e) = w;
        ps[l] = w;
        V.x(l, e) = make_float2(0.f, 0.f);
        s2 += w.x * w.x + w.y * w.y;
      } else {
        const float2 p = ps[l], s = V.s(l, e);
        pw += p.x * w.x + p.y * w.y;                    // Re(conj(pdir) w) = ||C pdir||^2
        sw += s.x * w.x + s.y * w.y;
        ww += w.x * w.x + w.y * w.y;
        s2 += s.x * s.x + s.y * s.y;
      }
    }
    lb += cnt;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      pw += __shfl_xor_sync(0xffffffffu, pw, o);
      sw += __shfl_xor_sync(0xffffffffu, sw, o);
      ww += __shfl_xor_sync(0xffffffffu, ww, o);
      s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    if ((g.tid & 31) == 0) red[g.tid >> 5] = make_float4(pw, sw, ww, s2);
    gsync(g);
    if (g.tid < int(G)) {
      float4 s = red[0];
#pragma unroll
      for (int i = 1; i < GT / 32; ++i) {
        const float4 q = red[i];
        s.x += q.x; s.y += q.y; s.z += q.z; s.w += q.w;
      }
      unsigned remote;
      asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(c.totals() + st)), "r"(unsigned(g.tid)));
      asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(remote), "f"(s.x), "f"(s.y), "f"(s.z), "f"(s.w) : "memory");
    }
    gsync(g);                                           // red is reused by the slot's next strip
  }
}
__device__ __forceinline__ float4 cg_totals(const Ctx& c, int n_strips) {   // after the team barrier: strips in order
  float4 s = c.totals()[0];
  for (int q = 1; q < n_strips; ++q) {
    const float4 r = c.totals()[q];
    s.x += r.x; s.y += r.y; s.z += r.z; s.w += r.w;
  }
  return s;
}
// x += alpha pdir, s -= alpha w, pdir = s + beta pdir on this slot's entries
__device__ __forceinline__ void cg_update(const Ctx& c, const Grp& g, const Vecs& V, float alpha, float beta) {
  float2* ps = c.ps(g.grp);
  for_own(*c.Lp(), g, [&](int l, int e) {
    const float2 p = ps[l], w = V.w(l, e);
    float2 x = V.x(l, e), s = V.s(l, e);
    x.x += alpha * p.x; x.y += alpha * p.y;
    s.x -= alpha * w.x; s.y -= alpha * w.y;
    V.x(l, e) = x;
    V.s(l, e) = s;
    ps[l] = make_float2(s.x + beta * p.x, s.y + beta * p.y);
  });
}

// ================================================================ decimated CG loop ("VR": vector-radix split of the grid)
// The mat-vecs of an iteration are cyclic correlations on the LED's mx x my grid.  Split the grid's SPATIAL side by the
// parity of (x, y) into four classes f_pq(x', y') = f(2x' + p, 2y' + q) of hx x hy = mx/2 x my/2 points.  With
// G_pq = DFT_{hx x hy} f_pq and Tw_pq(kx, ky) = W_mx^{p kx} W_my^{q ky}, the frequency side is reached by one radix-2 x 2
// butterfly per (kx, ky):
//     F(kx + a hx, ky + b hy) = sum_pq (-1)^{ap + bq} Tw_pq(kx, ky) G_pq(kx, ky),
//     f_pq = IDFT_{hx x hy} H_pq,      H_pq(kx, ky) = conj Tw_pq(kx, ky) sum_ab (-1)^{ap + bq} F(kx + a hx, ky + b hy).
// Everything that happens on the spatial side (the factors p_M, conj p_M) is pointwise, i.e. local to a class, and
// everything on the frequency side (scatter of pdir on U, the mask M_Q, the gather on U) is pointwise in (kx, ky) over the
// four classes.  So each CTA of a PAIR owns two classes (q = its cluster rank), keeps them and their p_M classes RESIDENT
// in shared memory, and runs "IDFT . p . DFT" as seven in-place shared-memory stages without leaving the SM; the pair
// meets only at the two frequency-side steps of an iteration, where each CTA publishes its G classes (82 KB, L2), passes
// ONE cluster barrier and reads the partner's.  An iteration costs 2 cluster barriers instead of 5 and no strip ever waits
// on L2; the CG vectors are kept redundantly by both CTAs (identical arithmetic on identical data, so alpha, beta and the
// stopping decision agree bit for bit).
// A class line of length L = 8 N2 (48, 64, 80, 96, 128) is transformed in two in-place stages, one sub-DFT per thread:
//   forward  s1: for n1 < 8: DFT_N2 over n2 of x[n1 + 8 n2], times W_L^{n1 k2}, stored at n1 + 8 k2
//            s2: for k2 < N2: DFT_8 over n1 of the 8 contiguous entries at 8 k2, stored at k1 + 8 k2  (= X[k2 + N2 k1])
//   inverse  s1': DFT_8^-1 over k1 of the entries at 8 k2, times conj W_L^{n1 k2};  s2': DFT_N2^-1 over k2, natural order out
// so the frequency side lives in the digit-swapped order s = k1 + 8 k2 <-> k = k2 + N2 k1 (the index tables are read
// through that map) and the spatial side in natural order.  Class rows have the odd pitch hx + 1 and threads map to lines
// first, so every access of every stage is a conflict-free 8-byte shared-memory access.
struct Vr {
  int hx, hy, P, csz, n2x, n2y;
  unsigned mag_nl, mag_hx;      // ceil(2^32 / (2 hy)), ceil(2^32 / hx): idx / d = umulhi(idx, mag) for idx d < 2^32
  bool p_smem;
};
__device__ __forceinline__ Vr vr_geometry(const DarkDev& L, const Ctx& c, int ng) {
  Vr v;
  v.hx = L.mx >> 1; v.hy = L.my >> 1; v.P = v.hx + 1; v.csz = v.hy * v.P;
  v.n2x = v.hx >> 3; v.n2y = v.hy >> 3;
  v.mag_nl = 0xFFFFFFFFu / unsigned(2 * v.hy) + 1u;
  v.mag_hx = 0xFFFFFFFFu / unsigned(v.hx) + 1u;
  v.p_smem = 4 * v.csz <= ng * (c.kex + c.kpc);
  return v;
}
// can this LED run the decimated loop?  (class lines of 8 x {6, 8, 10, 12, 16}; two T classes in the group regions; the
// exchange buffers in the tile's TM scratch; the redundant vectors in the CG region)
__device__ __forceinline__ bool vr_fits(const DarkDev& L, const Ctx& c, int ng, int vr_mu) {
  auto okl = [](int m) { return m == 96 || m == 128 || m == 160 || m == 192 || m == 256; };
  const int csz = (L.my >> 1) * ((L.mx >> 1) + 1);
  return okl(L.mx) && okl(L.my) && 2 * csz <= ng * (c.kex + c.kpc) && 8 * csz <= N * N && L.n_unknown <= vr_mu;
}

template <int N2, bool INV>
__device__ __forceinline__ void vr_load_strided(float2 (&v)[N2], const float2* e, int step) {
#pragma unroll
  for (int j = 0; j < N2; ++j) v[j] = e[j * step];
}
// rows, contiguous DFT_8 stage (inverse s1' / forward s2): sub-DFT (line l, k2)
template <bool INV>
__device__ __forceinline__ void vr_rows_c8(float2* T, const Vr& g, const float2* tw, int tid, int nt) {
  const int nl = 2 * g.hy;
  for (int idx = tid; idx < nl * g.n2x; idx += nt) {
    const int k2 = __umulhi(unsigned(idx), g.mag_nl), l = idx - k2 * nl;
    float2* e = T + l * g.P + 8 * k2;
    float2 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = e[j];
    RegDft<8, INV>::run(v);
    if (INV) {
#pragma unroll
      for (int j = 1; j < 8; ++j) v[j] = twmul<true>(v[j], tw[j + 8 * k2]);
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) e[j] = v[j];
  }
}
// rows, strided DFT_N2 stage (inverse s2' / forward s1): sub-DFT (line l, n1)
template <int N2, bool INV>
__device__ __forceinline__ void vr_rows_sn(float2* T, const Vr& g, const float2* tw, int tid, int nt) {
  const int nl = 2 * g.hy;
  for (int idx = tid; idx < nl * 8; idx += nt) {
    const int n1 = __umulhi(unsigned(idx), g.mag_nl), l = idx - n1 * nl;
    float2* e = T + l * g.P + n1;
    float2 v[N2];
#pragma unroll
    for (int j = 0; j < N2; ++j) v[j] = e[8 * j];
    RegDft<N2, INV>::run(v);
    if (!INV) {
#pragma unroll
      for (int j = 1; j < N2; ++j) v[j] = twmul<false>(v[j], tw[n1 + 8 * j]);
    }
#pragma unroll
    for (int j = 0; j < N2; ++j) e[8 * j] = v[j];
  }
}
// columns, contiguous DFT_8 stage: sub-DFT (class, column x', k2)
template <bool INV>
__device__ __forceinline__ void vr_cols_c8(float2* T, const Vr& g, const float2* tw, int tid, int nt) {
  for (int idx = tid; idx < 2 * g.hx * g.n2y; idx += nt) {
    const int r = __umulhi(unsigned(idx), g.mag_hx), x = idx - r * g.hx, k2 = r >> 1;
    float2* e = T + (r & 1) * g.csz + (8 * k2) * g.P + x;
    float2 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = e[j * g.P];
    RegDft<8, INV>::run(v);
    if (INV) {
#pragma unroll
      for (int j = 1; j < 8; ++j) v[j] = twmul<true>(v[j], tw[j + 8 * k2]);
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) e[j * g.P] = v[j];
  }
}
// columns, the middle stage: inverse s2' (natural order out), times p_M or conj p_M, forward s1: sub-DFT (class, x', n1).
// `pm` = this CTA's p_M classes in the layout of T (shared memory), or nullptr: read them from PF (global, natural grid).
template <int N2, bool CONJ>
__device__ __forceinline__ void vr_cols_mid(float2* T, const Vr& g, const float2* tw, const float2* pm, const float2* pf, int mx,
                                            int q, int tid, int nt) {
  for (int idx = tid; idx < 2 * g.hx * 8; idx += nt) {
    const int r = __umulhi(unsigned(idx), g.mag_hx), x = idx - r * g.hx, n1 = r >> 1, cl = r & 1;
    const int off = cl * g.csz + n1 * g.P + x;
    float2* e = T + off;
    float2 v[N2];
#pragma unroll
    for (int j = 0; j < N2; ++j) v[j] = e[(8 * j) * g.P];
    RegDft<N2, true>::run(v);
    if (pm) {
      const float2* pp = pm + off;
#pragma unroll
      for (int j = 0; j < N2; ++j) {
        const float2 p = pp[(8 * j) * g.P];
        v[j] = CONJ ? cmulc(v[j], p) : cmul(v[j], p);
      }
    } else {
      const float2* pp = pf + (2 * n1 + q) * mx + 2 * x + cl;   // natural point (2 x' + p, 2 (n1 + 8 j) + q)
#pragma unroll
      for (int j = 0; j < N2; ++j) {
        const float2 p = __ldcg(&pp[(16 * j) * mx]);
        v[j] = CONJ ? cmulc(v[j], p) : cmul(v[j], p);
      }
    }
    RegDft<N2, false>::run(v);
#pragma unroll
    for (int j = 1; j < N2; ++j) v[j] = twmul<false>(v[j], tw[n1 + 8 * j]);
#pragma unroll
    for (int j = 0; j < N2; ++j) e[(8 * j) * g.P] = v[j];
  }
}
#define WD_N2_SWITCH(n2, ...)                                  \
  switch (n2) {                                                \
    case 6: { constexpr int R = 6; __VA_ARGS__; } break;       \
    case 8: { constexpr int R = 8; __VA_ARGS__; } break;       \
    case 10: { constexpr int R = 10; __VA_ARGS__; } break;     \
    case 12: { constexpr int R = 12; __VA_ARGS__; } break;     \
    default: { constexpr int R = 16; __VA_ARGS__; } break;     \
  }
// IDFT_{hx x hy} . (conj) p_M . DFT_{hx x hy} on this CTA's two classes, in place (frequency side in, frequency side out)
template <bool CONJ>
__device__ __noinline__ void vr_local(float2* T, const Vr g, const float2* txs, const float2* tys, const float2* pm,
                                      const float2* pf, int mx, int q, int nt) {
  const int tid = threadIdx.x;
  vr_rows_c8<true>(T, g, txs, tid, nt);
  __syncthreads();
  WD_N2_SWITCH(g.n2x, vr_rows_sn<R, true>(T, g, txs, tid, nt));
  __syncthreads();
  vr_cols_c8<true>(T, g, tys, tid, nt);
  __syncthreads();
  WD_N2_SWITCH(g.n2y, vr_cols_mid<R, CONJ>(T, g, tys, pm, pf, mx, q, tid, nt));
  __syncthreads();
  vr_cols_c8<false>(T, g, tys, tid, nt);
  __syncthreads();
  WD_N2_SWITCH(g.n2x, vr_rows_sn<R, false>(T, g, txs, tid, nt));
  __syncthreads();
  vr_rows_c8<false>(T, g, txs, tid, nt);
  __syncthreads();
}

// The frequency-side step.  MODE 0: scatter pdir on U (no G input); 1: G -> F, keep Q, scale; 2: G -> F, gather U into w.
// Modes 0 / 1 leave H of this CTA's classes in T.  gx = the partner's published classes (global), q = cluster rank.
template <int MODE>
__device__ __noinline__ void vr_freq(float2* T, const Vr g, const DarkDev* Lp, const float2* wx, const float2* wy,
                                     const float2* gx, const float2* ps, float2* ws, int q, float scale, int nt) {
  const DarkDev& L = *Lp;
  const int mx = L.mx;
  for (int idx = threadIdx.x; idx < g.hx * g.hy; idx += nt) {
    const int sy = __umulhi(unsigned(idx), g.mag_hx), sx = idx - sy * g.hx;
    const int kx = (sx >> 3) + g.n2x * (sx & 7), ky = (sy >> 3) + g.n2y * (sy & 7);
    const int o = sy * g.P + sx;
    const float2 twx = wx[kx], twy = wy[ky];
    float2 f00, f10, f01, f11;                         // F(kx + a hx, ky + b hy) as f{a}{b}
    const int t00 = ky * mx + kx, t10 = t00 + g.hx, t01 = t00 + g.hy * mx, t11 = t01 + g.hx;
    if (MODE == 0) {
      auto at = [&](int t) {
        const int e = __ldg(&L.dmap_m[t]);
        return unsigned(e) < unsigned(L.n_unknown) ? ps[e] : make_float2(0.f, 0.f);
      };
      f00 = at(t00); f10 = at(t10); f01 = at(t01); f11 = at(t11);
    } else {
      // class (p, q'): own classes (q' = q) from T, the partner's from gx; local class index = p
      const float2 own0 = T[o], own1 = T[g.csz + o];
      const float2 oth0 = __ldcg(&gx[o]), oth1 = __ldcg(&gx[g.csz + o]);
      const float2 g00 = q ? oth0 : own0, g10r = q ? oth1 : own1, g01r = q ? own0 : oth0, g11r = q ? own1 : oth1;
      const float2 g10 = cmul(g10r, twx), g01 = cmul(g01r, twy), g11 = cmul(cmul(g11r, twx), twy);
      const float2 s0 = cadd(g00, g10), d0 = csub(g00, g10), s1 = cadd(g01, g11), d1 = csub(g01, g11);
      f00 = cadd(s0, s1); f10 = cadd(d0, d1); f01 = csub(s0, s1); f11 = csub(d0, d1);
    }
    if (MODE == 2) {
      auto put = [&](int t, float2 f) {
        const int e = __ldg(&L.dmap_m[t]);
        if (unsigned(e) < unsigned(L.n_unknown)) ws[e] = cscale(f, scale);
      };
      put(t00, f00); put(t10, f10); put(t01, f01); put(t11, f11);
      continue;
    }
    if (MODE == 1) {
      auto keep = [&](int t, float2 f) { return __ldg(&L.qmask_m[t]) ? cscale(f, scale) : make_float2(0.f, 0.f); };
      f00 = keep(t00, f00); f10 = keep(t10, f10); f01 = keep(t01, f01); f11 = keep(t11, f11);
    }
    // H_pq = conj Tw_pq sum_ab (-1)^{ap + bq} F_ab for q = this CTA's rank, p = 0, 1
    const float2 a0 = q ? csub(f00, f01) : cadd(f00, f01), a1 = q ? csub(f10, f11) : cadd(f10, f11);
    float2 h0 = cadd(a0, a1), h1 = cmulc(csub(a0, a1), twx);
    if (q) { h0 = cmulc(h0, twy); h1 = cmulc(h1, twy); }
    T[o] = h0;
    T[g.csz + o] = h1;
  }
}
// this CTA's classes -> the exchange buffer (16-byte copies; csz is even)
__device__ __forceinline__ void vr_publish(const float2* T, float2* dst, int csz, int nt) {
  const float4* s = reinterpret_cast<const float4*>(T);
  float4* d = reinterpret_cast<float4*>(dst);
  for (int i = threadIdx.x; i < csz; i += nt) d[i] = s[i];   // 2 classes x csz float2 = csz float4
}
// sum over the CTA of two values, identical in every thread (and in both CTAs: same data, same order)
__device__ __forceinline__ float2 vr_block_sum2(float a, float b, float2* red, int nwarps) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = make_float2(a, b);
  __syncthreads();
  float2 s = red[0];
  for (int i = 1; i < nwarps; ++i) { s.x += red[i].x; s.y += red[i].y; }
  return s;
}

// The CG loop of one LED on the decimated grid.  In: s0 = C^H d in `s0g` (global, all entries).  Out: x in the shared
// vector xs (both CTAs hold all of it).  Returns the iteration count.
template <int NG>
__device__ __noinline__ int vr_cg(const Args& a, const Ctx c, unsigned cr, float2* tm_t, const float2* pf_t, const float2* s0g,
                                  double& flop, bool mark, int& tl_n) {
#ifdef APIC_TIMELINE
#define VR_MARK(id)                                                                                   \
  do {                                                                                                \
    if (mark && threadIdx.x == 0 && tl_n + 1 < kTlCap) {                                              \
      unsigned long long t_;                                                                          \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                                          \
      a.tl[(size_t(cr) * NG) * kTlCap + ++tl_n] = (t_ << 8) | unsigned(id);                           \
    }                                                                                                 \
  } while (0)
#else
#define VR_MARK(id) do {} while (0)
#endif
  constexpr int NT = NG * GT;
  const DarkDev& L = *c.Lp();
  const Vr g = vr_geometry(L, c, NG);
  const int tid = threadIdx.x, q = int(cr), nu = L.n_unknown, mu = a.vr_mu;
  float2* T = c.base();
  float2* pm = g.p_smem ? T + 2 * g.csz : nullptr;
  float2 *txs = c.twx(), *wx = c.twx() + 128, *tys = c.twy(), *wy = c.twy() + 128;
  float2 *ws = c.cg(0), *ss = ws + mu, *ps = ss + mu, *xs = ps + mu;
  float2* red = reinterpret_cast<float2*>(c.red(0));
  const float scale = 1.f / float(L.mx * L.my);
  // tables: stage twiddles W_L^{n1 k2} at [n1 + 8 k2], butterfly twiddles W_mx^{kx}, W_my^{ky}
  if (tid < 128) {
    const int n1 = tid & 7, k2 = tid >> 3;
    float sn, cs;
    sincospif(-2.f * float((n1 * k2) % g.hx) / float(g.hx), &sn, &cs);
    txs[tid] = make_float2(cs, sn);
    sincospif(-2.f * float((n1 * k2) % g.hy) / float(g.hy), &sn, &cs);
    tys[tid] = make_float2(cs, sn);
  } else if (tid < 256) {
    const int k = tid - 128;
    float sn, cs;
    sincospif(-2.f * float(k) / float(L.mx), &sn, &cs);
    wx[k] = make_float2(cs, sn);
    sincospif(-2.f * float(k) / float(L.my), &sn, &cs);
    wy[k] = make_float2(cs, sn);
  }
  // p_M classes of this CTA (rows of parity q): class p at pm + p csz
  if (pm) {
    for (int y = tid >> 5; y < g.hy; y += NT / 32) {
      const float2* src = pf_t + (2 * y + q) * L.mx;
      for (int X = tid & 31; X < L.mx; X += 32) pm[(X & 1) * g.csz + y * g.P + (X >> 1)] = __ldcg(&src[X]);
    }
  }
  float gs = 0.f;
  for (int e = tid; e < nu; e += NT) {
    const float2 s = __ldcg(&s0g[e]);
    ss[e] = s; ps[e] = s; xs[e] = make_float2(0.f, 0.f);
    gs += s.x * s.x + s.y * s.y;
  }
  float gamma = vr_block_sum2(gs, 0.f, red, NT / 32).x;   // also orders the table / vector writes before their use
  const float gamma0 = gamma;
  int iters = 0, buf = 0;
  bool done = !(gamma > 0.f);
  const double fl_iter = 2.0 * (2.0 * (2 * g.hy) * line_flop(g.hx) + 2.0 * (2 * g.hx) * line_flop(g.hy));
  VR_MARK(40);
  while (!done && iters < a.max_iters) {
    VR_MARK(41);
    vr_freq<0>(T, g, &L, wx, wy, nullptr, ps, nullptr, q, scale, NT);
    __syncthreads();
    VR_MARK(42);
    vr_local<true>(T, g, txs, tys, pm, pf_t, L.mx, q, NT);
    VR_MARK(43);
    vr_publish(T, tm_t + (buf * 4 + 2 * q) * g.csz, g.csz, NT);
    VR_MARK(44);
    team_sync(true);
    VR_MARK(45);
    vr_freq<1>(T, g, &L, wx, wy, tm_t + (buf * 4 + 2 * (1 - q)) * g.csz, nullptr, nullptr, q, scale, NT);
    buf ^= 1;
    __syncthreads();
    VR_MARK(46);
    vr_local<false>(T, g, txs, tys, pm, pf_t, L.mx, q, NT);
    VR_MARK(47);
    vr_publish(T, tm_t + (buf * 4 + 2 * q) * g.csz, g.csz, NT);
    VR_MARK(48);
    team_sync(true);
    VR_MARK(49);
    vr_freq<2>(T, g, &L, wx, wy, tm_t + (buf * 4 + 2 * (1 - q)) * g.csz, nullptr, ws, q, scale, NT);
    buf ^= 1;
    __syncthreads();
    VR_MARK(50);
    if (tid == 0) flop += fl_iter;
    ++iters;
    // plain CG update, redundantly in both CTAs (df_mgrid.cu's cg_update)
    float pw = 0.f;
    for (int e = tid; e < nu; e += NT) pw += ps[e].x * ws[e].x + ps[e].y * ws[e].y;   // Re(conj(pdir) w) = ||C pdir||^2
    pw = vr_block_sum2(pw, 0.f, red, NT / 32).x;
    if (!(pw > 0.f)) break;
    const float alpha = gamma / pw;
    float gsum = 0.f;
    for (int e = tid; e < nu; e += NT) {
      const float2 p = ps[e], w = ws[e];
      float2 x = xs[e], s = ss[e];
      x.x += alpha * p.x; x.y += alpha * p.y;
      s.x -= alpha * w.x; s.y -= alpha * w.y;
      xs[e] = x; ss[e] = s;
      gsum += s.x * s.x + s.y * s.y;
    }
    gsum = vr_block_sum2(gsum, 0.f, red, NT / 32).x;
    const float beta = gsum / gamma;
    for (int e = tid; e < nu; e += NT) {
      const float2 s = ss[e], p = ps[e];
      ps[e] = make_float2(s.x + beta * p.x, s.y + beta * p.y);
    }
    gamma = gsum;
    done = !(gsum > a.tol2 * gamma0);
    __syncthreads();
    VR_MARK(51);
  }
  return iters;
}

// ================================================================ the kernel
// MINB = CTAs per SM the kernel is compiled for (register cap 64K / (NG * 256 * MINB)): NG * MINB = 4 is the 64-register
// wide shape; NG = 1, MINB = 2 is df_mgrid.cu's shape (128 registers, 2 CTAs of 256 threads per SM) with this file's data path
template <int NG, int MINB>
__global__ void __launch_bounds__(NG * GT, MINB) df_wide_kernel(const __grid_constant__ Args a) {
  Ctx c;
  c.kex = a.kex; c.kpc = a.kpc; c.cap = a.cap; c.ng = NG;
  c.nvec = 4 - ((a.vec_global & 1) + (a.vec_global >> 1 & 1) + (a.vec_global >> 2 & 1));
  float2* tws = c.twx();                               // [3][256]: rows, columns, N grid
  float* c_sh = c.c_sh();
  DarkDev& Lsh = *c.Lp();
  const unsigned G = cluster_size(), cr = cluster_rank();
  const bool multi = G > 1;
  Grp g;
  g.tid = int(threadIdx.x) & (GT - 1);
  g.grp = int(threadIdx.x) / GT;
  g.S = int(G) * NG;
  g.sigma = g.grp * int(G) + int(cr);                  // consecutive strips go to different CTAs first
  const int team_id = blockIdx.x / G, n_teams = gridDim.x / G;
  if (threadIdx.x < 256) tws[512 + threadIdx.x] = a.t.tw_xy[4 * 256 + threadIdx.x];
  const int live_n = *a.live_count - a.chunk0;
  const int tiles = live_n < a.n_tiles ? live_n : a.n_tiles;
  const int nz = a.t.nz;
  double flop = 0.0;
  int tl_n = 0;
  auto mine = [&](int n_st) { return (n_st > g.sigma) ? (n_st - g.sigma + g.S - 1) / g.S : 0; };

  for (int slot = team_id; slot < tiles; slot += n_teams) {
    const int tile = a.live[a.chunk0 + slot];
    float2* const o_t = a.O + size_t(slot) * (N * N);   // this tile's object spectrum and scratch grids
    float2* const tn_t = a.T + size_t(slot) * (N * N);
    float2* const tm_t = a.TM + size_t(slot) * (N * N);
    float2* const pf_t = a.PF + size_t(slot) * (N * N);
    Vecs V;                                              // where this slot's w, s, x live
    {
      float2* sm = c.cg(g.grp) + c.cap;
      const size_t go = size_t(slot) * a.max_unknown;
      V.w.gl = a.vec_global & 1; V.w.p = V.w.gl ? a.VW + go : sm; if (!V.w.gl) sm += c.cap;
      V.s.gl = a.vec_global >> 1 & 1; V.s.p = V.s.gl ? a.VS + go : sm; if (!V.s.gl) sm += c.cap;
      V.x.gl = a.vec_global >> 2 & 1; V.x.p = V.x.gl ? a.VX + go : sm;
    }
    __syncthreads();
    if (threadIdx.x < nz) c_sh[threadIdx.x] = a.coef[size_t(slot) * nz + threadIdx.x];
    for (int k = 0; k < a.n_leds; ++k) {
      __syncthreads();
      if (threadIdx.x < sizeof(DarkDev) / sizeof(int))
        reinterpret_cast<int*>(&Lsh)[threadIdx.x] = reinterpret_cast<const int*>(&a.leds[k])[threadIdx.x];
      __syncthreads();
      const int r1x = Lsh.mx >> 4, r1y = Lsh.my >> 4;
      if (threadIdx.x < 256) {
        tws[threadIdx.x] = a.t.tw_xy[tw_slot(r1x) * 256 + threadIdx.x];
        tws[256 + threadIdx.x] = a.t.tw_xy[tw_slot(r1y) * 256 + threadIdx.x];
      }
      const int n_d = (Lsh.d_nrow + 15) >> 4, n_q = (Lsh.q_nrow + 15) >> 4, n_u = (Lsh.u_nrow + 15) >> 4, n_c = Lsh.mx >> 4;
      if (g.sigma < n_q) { WD_R1_SWITCH(r1x, c.kq(g.grp)[g.tid] = q_keep_bits<R>(Lsh, g.sigma, g.tid)); }
      __syncthreads();
      // ---- setup: P_hat -> p_N, p_M -> d on Q -> s = C^H d
      WD_MARK(100 + k);
      ph_build_p_rows_n(c, g, o_t, tn_t, nz);
      WD_R1_SWITCH(r1x, ph_build_p_rows_m<R>(c, g, o_t, tm_t, nz));
      WD_MARK(20);
      team_sync(multi);
      WD_MARK(21);
      ph_cols_rhs_n(c, g, tn_t, a.src, size_t(tile) * a.t.n_img + a.t.nb + Lsh.led);
      WD_R1_SWITCH(r1y, ph_cols_pm<R>(c, g, tm_t, pf_t));
      WD_MARK(22);
      team_sync(multi);
      WD_MARK(23);
      WD_R1_SWITCH(r1x, ph_rows_rhs<R>(c, g, tn_t, tm_t));
      WD_MARK(24);
      team_sync(multi);
      WD_MARK(25);
      WD_R1_SWITCH(r1y, ph_cols_mul<R, false>(c, g, tm_t, pf_t, true));
      WD_MARK(26);
      team_sync(multi);
      WD_MARK(27);
      WD_R1_SWITCH(r1x, ph_rows_u_gather<R>(c, g, tm_t, V.w));
      cg_partials(c, g, V, true, G);
      WD_MARK(28);
      team_sync(multi);
      WD_MARK(29);
      if (g.tid == 0) {
        const double fx = 16.0 * line_flop(Lsh.mx), fy = 16.0 * line_flop(Lsh.my), fn = 16.0 * line_flop(N);
        flop += mine(n_d) * (fn + fx) + mine(N / 16) * 2 * fn + mine(n_c) * fy + mine(n_q) * (fn + fx) + mine(n_c) * 2 * fy +
                mine(n_u) * fx;
      }
      int iters = 0;
      const bool use_vr = NG == 4 && a.vr && G == 2 && vr_fits(Lsh, c, NG, a.vr_mu);   // compiled into the 1024-thread shape only
      if (use_vr) {
        // s0 = C^H d sits in VW (global; the wide set-up wrote it before the barrier above): both CTAs take all of it
        iters = vr_cg<NG>(a, c, cr, tm_t, pf_t, V.w.p, flop, a.tl && team_id == 0, tl_n);
        WD_MARK(52);
        // ---- S10 from the shared x (both CTAs hold all entries; they split them)
        const float2* xs = c.cg(0) + 3 * a.vr_mu;
        for (int e = int(cr) * (NG * GT) + threadIdx.x; e < Lsh.n_unknown; e += 2 * NG * GT) {
          const float phi = zern_phase(Lsh.zern + size_t(e) * nz, c_sh, nz);
          float sn, cs;
          sincosf(phi, &sn, &cs);
          const int q = Lsh.disc_f[e];
          const float2 u = cmulc(xs[e], make_float2(cs, sn));
          o_t[q] = Lsh.accumulate ? cadd(__ldcg(&o_t[q]), u) : u;
        }
        if (g.sigma == 0 && g.tid == 0) a.cg_iters[size_t(slot) * a.n_leds + k] = iters;
      } else {
      const float gamma0 = cg_totals(c, n_u).w;
      bool done = !(gamma0 > 0.f);
      // ---- CG on the normal equations
      while (!done && iters < a.max_iters) {
        gsync(g);                                          // pdir of this slot complete in shared memory
        WD_MARK(1);
        WD_R1_SWITCH(r1x, ph_rows_u_scatter<R>(c, g, tm_t));
        WD_MARK(2);
        team_sync(multi);
        WD_MARK(3);
        WD_R1_SWITCH(r1y, ph_cols_mul<R, true>(c, g, tm_t, pf_t, false));
        WD_MARK(4);
        team_sync(multi);
        WD_MARK(5);
        WD_R1_SWITCH(r1x, ph_rows_q<R>(c, g, tm_t));
        WD_MARK(6);
        team_sync(multi);
        WD_MARK(7);
        WD_R1_SWITCH(r1y, ph_cols_mul<R, false>(c, g, tm_t, pf_t, false));
        WD_MARK(8);
        team_sync(multi);
        WD_MARK(9);
        WD_R1_SWITCH(r1x, ph_rows_u_gather<R>(c, g, tm_t, V.w));
        cg_partials(c, g, V, false, G);
        WD_MARK(10);
        team_sync(multi);
        WD_MARK(11);
        ++iters;
        const float4 tot = cg_totals(c, n_u);              // <pdir, w>, <s, w>, <w, w>, <s, s>
        if (!(tot.x > 0.f)) break;
        const float gamma = tot.w, alpha = gamma / tot.x;
        const float gnew = fmaxf(gamma - 2.f * alpha * tot.y + alpha * alpha * tot.z, 0.f);   // ||s - alpha w||^2
        cg_update(c, g, V, alpha, gnew / gamma);
        WD_MARK(12);
        done = !(gnew > a.tol2 * gamma0);
      }
      if (g.tid == 0)                                      // executed line transforms of the loop (nothing of this is live inside it)
        flop += double(iters) * (2 * mine(n_u) * 16.0 * line_flop(Lsh.mx) + 4 * mine(n_c) * 16.0 * line_flop(Lsh.my) +
                                 2 * mine(n_q) * 16.0 * line_flop(Lsh.mx));
      gsync(g);
      // ---- S10: O_hat(u) = U_hat(u) e^{-j phi(u+kappa)}, known ∪= U (every slot extends with its share)
      {
        for_own(Lsh, g, [&](int l, int e) {
          const float phi = zern_phase(Lsh.zern + size_t(e) * nz, c_sh, nz);
          float sn, cs;
          sincosf(phi, &sn, &cs);
          const int q = Lsh.disc_f[e];
          const float2 u = cmulc(V.x(l, e), make_float2(cs, sn));
          o_t[q] = Lsh.accumulate ? cadd(__ldcg(&o_t[q]), u) : u;   // ring-wise order (R15b): sum now, mean at the end of the ring
        });
        if (g.sigma == 0 && g.tid == 0) a.cg_iters[size_t(slot) * a.n_leds + k] = iters;
      }
      }
      team_sync(multi);                                    // O complete before the next LED reads it
      if (Lsh.n_avg > 0) {                                 // df_order 1, end of a ring: bins solved by c LEDs hold a sum of c solutions
        for (int i = int(cr) * (NG * GT) + threadIdx.x; i < Lsh.n_avg; i += int(G) * (NG * GT)) {
          const int q = __ldg(&Lsh.avg_f[i]);
          o_t[q] = cscale(__ldcg(&o_t[q]), __ldg(&Lsh.avg_w[i]));
        }
        team_sync(multi);
      }
    }
  }
  if (g.tid == 0 && flop > 0.0) atomicAdd(a.work, (unsigned long long)(flop + 0.5));
}

// Developer knobs (APIC_DF_NO_VR, APIC_DF_WIDE_DEBUG, APIC_DF_TIMELINE, APIC_DF_WIDE_NG) exist only in a build with
// APIC_EXTRA_NVCC_FLAGS=-DAPIC_DF_KNOBS (or -DAPIC_TIMELINE); the shipped library reads no environment variable.  Read
// once per process.
#if defined(APIC_DF_KNOBS) || defined(APIC_TIMELINE)
static const char* knob(int which) {
  static const char* const v[4] = {getenv("APIC_DF_NO_VR"), getenv("APIC_DF_WIDE_DEBUG"), getenv("APIC_DF_TIMELINE"),
                                   getenv("APIC_DF_WIDE_NG")};
  return v[which];
}
#else
static constexpr const char* knob(int) { return nullptr; }
#endif
enum { KNOB_NO_VR = 0, KNOB_DEBUG = 1, KNOB_TIMELINE = 2, KNOB_NG = 3 };

// cudaFuncSetAttribute is per device and per kernel instantiation: done when the shared-memory size first grows past
// what was set (device, instantiation) - not on every pass of the hot path.
template <int NG, int MINB>
static bool ensure_attributes(int device, size_t smem) {
  constexpr int kMaxDev = 64;
  static size_t set_smem[kMaxDev] = {};
  static std::mutex mu;
  if (device < 0 || device >= kMaxDev) return false;
  std::lock_guard<std::mutex> lock(mu);
  if (set_smem[device] >= smem && set_smem[device] != 0) return true;
  auto kern = df_wide_kernel<NG, MINB>;
  const cudaError_t e1 = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
  const cudaError_t e2 = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e1 != cudaSuccess || e2 != cudaSuccess) {
    if (knob(KNOB_DEBUG)) fprintf(stderr, "df_wide: attr %s / %s\n", cudaGetErrorString(e1), cudaGetErrorString(e2));
    cudaGetLastError();
    return false;
  }
  set_smem[device] = smem;
  return true;
}

template <int NG, int MINB>
static bool launch_ng(const Args& a0, const DarkDev* h_leds, int n_leds, const LaunchCtx& c, int G, int sms) {
  Args a = a0;
  if (G < 1) G = 1;
  while (G * NG > kMaxSlots) --G;
  const int S = G * NG;
  // a slot's share of the CG vectors: the entries of the U-row strips sigma, sigma + S, ... (largest over LEDs and slots)
  int cap = 2;
  for (int k = 0; k < n_leds; ++k) {
    const int n_u = (h_leds[k].u_nrow + 15) >> 4;
    for (int sg = 0; sg < S; ++sg) {
      int s = 0;
      for (int st = sg; st < n_u; st += S) s += h_leds[k].u_strip_off[st + 1] - h_leds[k].u_strip_off[st];
      cap = std::max(cap, s);
    }
  }
  a.cap = (cap + 1) & ~1;
  // pdir always in shared memory; w, s, x as the 227 KB allow (else in global memory: L2-resident, touched once or twice per iteration)
  auto smem_for = [&](int nvec) { return (size_t(NG) * (a.kex + a.kpc) + kSmFixed + size_t(NG) * 128 + size_t(NG) * nvec * a.cap) * sizeof(float2); };
  int nvec = 4;
  while (nvec > 1 && smem_for(nvec) > size_t(227 * 1024)) --nvec;
  size_t smem = smem_for(nvec);
  a.vr = 0;
  if (NG == 4 && G == 2 && !knob(KNOB_NO_VR)) {
    // decimated CG loop: w of the set-up in global memory, the CG region holds four redundant vectors of max_unknown
    int mu = 2;
    for (int k = 0; k < n_leds; ++k) mu = std::max(mu, h_leds[k].n_unknown);
    mu = (mu + 1) & ~1;
    const size_t cgreg = std::max(size_t(NG) * a.cap, size_t(4) * mu);
    const size_t sm = (size_t(NG) * (a.kex + a.kpc) + kSmFixed + size_t(NG) * 128 + cgreg) * sizeof(float2);
    if (sm <= size_t(227 * 1024)) { a.vr = 1; a.vr_mu = mu; nvec = 1; smem = sm; }
  }
  a.vec_global = nvec == 4 ? 0 : nvec == 3 ? 4 : nvec == 2 ? 6 : 7;
  const bool dbg = knob(KNOB_DEBUG) != nullptr;
  if (dbg) fprintf(stderr, "df_wide: NG %d G %d kex %d kpc %d cap %d smem %zu\n", NG, G, a.kex, a.kpc, a.cap, smem);
  if (dbg) fprintf(stderr, "df_wide: vec_global %d\n", a.vec_global);
  if (smem > size_t(227 * 1024)) return false;
  auto kern = df_wide_kernel<NG, MINB>;
  if (!ensure_attributes<NG, MINB>(c.pd->device, smem)) return false;   // nothing pending: the caller may fall back
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = unsigned(G); at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeClusterSchedulingPolicyPreference;
  at[1].val.clusterSchedulingPolicyPreference = cudaClusterSchedulingPolicyLoadBalancing;
  cfg.blockDim = dim3(NG * GT);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = c.stream;
  cfg.attrs = at;
  cfg.numAttrs = 2;
  int max_clusters = 0;
  cfg.gridDim = dim3(unsigned(G) * unsigned(std::max(1, sms / G)));
  {
    const cudaError_t e3 = cudaOccupancyMaxActiveClusters(&max_clusters, kern, &cfg);
    if (dbg) fprintf(stderr, "df_wide: max active clusters %d (%s)\n", max_clusters, cudaGetErrorString(e3));
    if (e3 != cudaSuccess || max_clusters < 1) {
      cudaGetLastError();
      return false;
    }
  }
  const int teams = std::max(1, std::min(max_clusters, c.chunk_tiles));
  cfg.gridDim = dim3(unsigned(G) * unsigned(teams));
  const char* tl_path = knob(KNOB_TIMELINE);
  const size_t tl_words = size_t(G) * NG * kTlCap;
  if (tl_path) {
    cudaMalloc(&a.tl, tl_words * sizeof(unsigned long long));
    cudaMemsetAsync(a.tl, 0, tl_words * sizeof(unsigned long long), c.stream);
  }
  bool ok;
  {
    ProfScope ps(c, CAT_DF_WIDE);
    ok = cudaLaunchKernelEx(&cfg, kern, a) == cudaSuccess;
  }
  // A failed launch enqueued nothing; clear its error so that the caller's fallback kernel is judged on its own.
  if (!ok) cudaGetLastError();
  if (tl_path) {                                         // debugging aid: marks of team 0, one line per mark: cta group ns id
    std::vector<unsigned long long> h(tl_words);
    cudaStreamSynchronize(c.stream);
    cudaMemcpy(h.data(), a.tl, h.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    cudaFree(a.tl);
    if (FILE* f = fopen(tl_path, "w")) {
      for (int q = 0; q < G * NG; ++q)
        for (int i = 1; i < kTlCap && h[size_t(q) * kTlCap + i]; ++i)
          fprintf(f, "%d %d %llu %llu\n", q / NG, q % NG, h[size_t(q) * kTlCap + i] >> 8, h[size_t(q) * kTlCap + i] & 255ull);
      fclose(f);
    }
  }
  return ok;
}

}  // namespace wd

// Returns false when the configuration does not fit (the caller falls back to df_mgrid.cu).
bool launch_darkfield_wide(const DevTables& t, const DarkDev* d_leds, const DarkDev* h_leds, int n_leds, const Workspace& w,
                           const LaunchCtx& c, const ImgSrc& src, int df_iters, float df_tol, int team_size, int groups) {
  using namespace wd;
  if (n_leds <= 0) return true;
  int r1max = 6, r1ymax = 6;
  for (int k = 0; k < n_leds; ++k) {
    r1max = std::max(r1max, std::max(h_leds[k].mx, h_leds[k].my) >> 4);
    r1ymax = std::max(r1ymax, h_leds[k].my >> 4);
  }
  Args a{};
  a.t = t; a.leds = d_leds; a.n_leds = n_leds; a.src = src; a.O = w.O; a.coef = w.coef; a.T = w.T; a.TM = w.TM;
  a.PF = w.PF; a.VW = w.vec_w; a.VS = w.vec_s; a.VX = w.vec_x; a.max_unknown = w.max_unknown; a.cg_iters = w.cg_iters; a.max_iters = df_iters; a.tol2 = df_tol * df_tol; a.live = c.live;
  a.live_count = c.live_count; a.chunk0 = c.chunk0; a.n_tiles = c.chunk_tiles; a.work = w.df_work;
  // exchange buffer: 16 lines x R1 x 18 padded entries (row type X, the largest of the layouts); p_M strip: 16 x my;
  // both together hold the 16 x 273 strip of the N-grid transforms
  a.kex = 16 * r1max * 18;
  a.kpc = 256 * r1ymax;
  if (a.kex + a.kpc < 16 * S256::LS) a.kex = 16 * S256::LS - a.kpc;
  a.kex = (a.kex + 1) & ~1;
  const int sms = c.pd->sms;
  int ng = groups > 0 ? groups : 4;   // 4, 2, 1: groups per CTA at 64 registers; 11: one group at 128 registers
  if (groups != 11)
    if (const char* e = knob(KNOB_NG)) ng = atoi(e);   // experiments with the shapes of mode 5 (-DAPIC_DF_KNOBS builds)
  int G = team_size;
  if (G <= 0) {
    // NG = 4: pairs of 1024-thread CTAs, one CTA per SM (the decimated CG loop needs exactly this shape; larger passes
    // loop over their tiles); NG = 2 / 1: as many CTAs per tile as the pass leaves resident slots for
    if (ng == 4) {
      G = 2;
    } else {
      // measured on config 2 with df_mgrid.cu's identical shape (ms per step): 32 tiles G = 8: 8.3; 56 tiles G = 5: 10.4;
      // 64 tiles G = 4: 12.1; cluster sizes 6 and 7 place badly and are skipped
      const int ctas = ng == 2 || ng == 11 ? 2 * sms : 4 * sms;
      G = 1;
      for (int cand : {8, 5, 4, 2})
        if (cand * c.chunk_tiles <= ctas) { G = cand; break; }
    }
  }
  switch (ng) {
    case 4: return launch_ng<4, 1>(a, h_leds, n_leds, c, G, sms);
    case 2: return launch_ng<2, 2>(a, h_leds, n_leds, c, G, sms);
    case 11: return launch_ng<1, 2>(a, h_leds, n_leds, c, G, sms);   // 128 registers
    default: return launch_ng<1, 4>(a, h_leds, n_leds, c, G, sms);
  }
}

}  // namespace apic
