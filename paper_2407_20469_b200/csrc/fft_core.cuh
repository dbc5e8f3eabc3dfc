// fft_core.cuh - batched shared-memory complex FFT building blocks (libapic kernel K1).
//
// Every transform of the APIC path (Eq. 5-7; Eq. 13 mat-vecs) is a
// 2-D DFT of an N x N tile, N in {64,128,256,512}, executed as 1-D "line" transforms over strips
// of LINES lines: a row strip (consecutive rows) or a column strip (consecutive columns, one
// 64/128-byte global segment per row).
//
// A line transform is a register-resident Cooley-Tukey FFT with N = R * B * R:
//     n = n1 + R n2 + R B n3,   k = k1 + R k2 + R B k3        (n1,n3,k1,k3 < R;  n2,k2 < B)
//   step 1  thread t = n1 + R n2 holds x[t + TPL r], r < R (TPL = N/R threads per line): DFT_R over
//           n3, twiddle, written IN PLACE to shared memory
//   step 2  (only if B > 1) thread (n1,k1): DFT_B over n2, twiddle, in place
//   step 3  thread t' = k1 + R k2 reads R contiguous values, DFT_R over n1 and holds X[t' + TPL r]
// so the output distribution over threads equals the input distribution: transforms chain through
// REGISTERS (IFFT -> pointwise -> FFT never touches shared memory in between), global loads feed
// step 1 directly and step 3 stores straight to global memory.  One line costs one write + one
// read of shared memory (two for N = 128, 512) and two (three) barriers; lines are padded
// (i + i/16, odd line stride) so that all strided accesses are bank-conflict free or 2-way.
// Natural order in and out, unnormalised:
//     forward  X[k] = sum_n x[n] e^{-2 pi i k n / N},    inverse  x[n] = sum_k X[k] e^{+2 pi i k n / N}.
// Twiddles come from fp64-computed tables (host: build_twiddles) laid out so that the threads of
// a half-warp read consecutive entries.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <vector>

namespace apic {

__host__ __device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__host__ __device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__host__ __device__ __forceinline__ float2 cmulc(float2 a, float2 b) {  // a * conj(b)
  return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__host__ __device__ __forceinline__ float2 cscale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }

// multiply by e^{-+ i pi/2}: forward (-i), inverse (+i)
template <bool INV>
__host__ __device__ __forceinline__ float2 rot90(float2 a) {
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}
// multiply by (c - i s) forward, (c + i s) inverse
template <bool INV>
__host__ __device__ __forceinline__ float2 rot(float2 a, float c, float s) {
  return INV ? make_float2(a.x * c - a.y * s, a.y * c + a.x * s)
             : make_float2(a.x * c + a.y * s, a.y * c - a.x * s);
}
// multiply by a table twiddle w = e^{-i phi} (forward) or its conjugate (inverse)
template <bool INV>
__host__ __device__ __forceinline__ float2 twmul(float2 a, float2 w) {
  return INV ? cmulc(a, w) : cmul(a, w);
}

// ---- register DFTs, natural order in/out: V[m] = sum_r v[r] e^{-+ 2 pi i r m / R}
template <bool INV>
__host__ __device__ __forceinline__ void dft4(float2& a, float2& b, float2& c, float2& d) {
  float2 t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = rot90<INV>(csub(b, d));
  a = cadd(t0, t2);
  b = cadd(t1, t3);
  c = csub(t0, t2);
  d = csub(t1, t3);
}

template <int R, bool INV>
struct RegDft;

template <bool INV>
struct RegDft<4, INV> {
  static __host__ __device__ __forceinline__ void run(float2 (&v)[4]) { dft4<INV>(v[0], v[1], v[2], v[3]); }
};

template <bool INV>
struct RegDft<8, INV> {
  static __host__ __device__ __forceinline__ void run(float2 (&v)[8]) {
    constexpr float h = 0.70710678118654752440f;
    float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    float2 o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
    dft4<INV>(e0, e1, e2, e3);
    dft4<INV>(o0, o1, o2, o3);
    o1 = rot<INV>(o1, h, h);          // w8^1
    o2 = rot90<INV>(o2);              // w8^2
    o3 = rot<INV>(o3, -h, h);         // w8^3
    v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
    v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
    v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
    v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
  }
};

template <bool INV>
struct RegDft<16, INV> {
  static __host__ __device__ __forceinline__ void run(float2 (&v)[16]) {
    constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;  // pi/8
    constexpr float h = 0.70710678118654752440f;
    float2 x[4][4];                        // X_b[m1] = DFT4 over a of v[4a+b]
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      x[b][0] = v[b]; x[b][1] = v[4 + b]; x[b][2] = v[8 + b]; x[b][3] = v[12 + b];
      dft4<INV>(x[b][0], x[b][1], x[b][2], x[b][3]);
    }
    x[1][1] = rot<INV>(x[1][1], c1, s1);   // w16^{b*m1}: e=1
    x[1][2] = rot<INV>(x[1][2], h, h);     // e=2
    x[1][3] = rot<INV>(x[1][3], s1, c1);   // e=3
    x[2][1] = rot<INV>(x[2][1], h, h);     // e=2
    x[2][2] = rot90<INV>(x[2][2]);         // e=4
    x[2][3] = rot<INV>(x[2][3], -h, h);    // e=6
    x[3][1] = rot<INV>(x[3][1], s1, c1);   // e=3
    x[3][2] = rot<INV>(x[3][2], -h, h);    // e=6
    x[3][3] = rot<INV>(x[3][3], -c1, -s1); // e=9
#pragma unroll
    for (int m1 = 0; m1 < 4; ++m1) {       // V[m1 + 4 m2] = DFT4 over b of X_b[m1]
      float2 y0 = x[0][m1], y1 = x[1][m1], y2 = x[2][m1], y3 = x[3][m1];
      dft4<INV>(y0, y1, y2, y3);
      v[m1] = y0; v[m1 + 4] = y1; v[m1 + 8] = y2; v[m1 + 12] = y3;
    }
  }
};

// ---- per-N factorisation N = R * B * R and strip shape
template <int N> struct FftCfg;
// MINB = CTAs per SM the strip kernels are compiled for (register cap = 64K / (THREADS * MINB))
template <> struct FftCfg<64>  { static constexpr int R = 8,  B = 1, LINES = 16, MINB = 8; };
template <> struct FftCfg<128> { static constexpr int R = 4,  B = 8, LINES = 8,  MINB = 4; };
template <> struct FftCfg<256> { static constexpr int R = 16, B = 1, LINES = 16, MINB = 4; };
template <> struct FftCfg<512> { static constexpr int R = 8,  B = 8, LINES = 8,  MINB = 2; };

// LINES_ lines per strip (default: the per-N value of FftCfg; the darkfield team kernel uses wider strips)
template <int N, int LINES_ = FftCfg<N>::LINES>
struct Strip {
  using C = FftCfg<N>;
  static constexpr int R = C::R, B = C::B, LINES = LINES_, MINB = C::MINB;
  static constexpr int TPL = N / R;                 // threads per line
  static constexpr int THREADS = LINES * TPL;
  static constexpr int LS = N + N / 16 + 1;         // padded line stride (odd)
  static constexpr size_t SMEM = size_t(LINES) * LS * sizeof(float2);
  static constexpr int TW_ENTRIES = (B == 1) ? R * R : R * B + B * R * R;
};

inline int strip_lines(int n) { return n == 64 ? 16 : n == 128 ? 8 : n == 256 ? 16 : 8; }

// Host: twiddle tables e^{-2 pi i m / N} in the layouts the steps read.
//   B == 1 : tw[k1 * R + n1]                     = W_N^{n1 k1}
//   B  > 1 : tw[k1 * B + n2]                     = W_N^{R n2 k1}        (after step 1)
//            tw[R*B + k2 * R*R + (n1 + R k1)]    = W_N^{n1 (k1 + R k2)} (after step 2)
template <int N>
inline void build_twiddles_n(std::vector<float2>& tw) {
  constexpr int R = Strip<N>::R, B = Strip<N>::B;
  auto w = [](long long m) {
    const double a = -2.0 * M_PI * double(m % N) / double(N);
    return make_float2(float(std::cos(a)), float(std::sin(a)));
  };
  tw.assign(Strip<N>::TW_ENTRIES, make_float2(1.f, 0.f));
  if (B == 1) {
    for (int k1 = 0; k1 < R; ++k1)
      for (int n1 = 0; n1 < R; ++n1) tw[k1 * R + n1] = w((long long)n1 * k1);
  } else {
    for (int k1 = 0; k1 < R; ++k1)
      for (int n2 = 0; n2 < B; ++n2) tw[k1 * B + n2] = w((long long)R * n2 * k1);
    for (int k2 = 0; k2 < B; ++k2)
      for (int k1 = 0; k1 < R; ++k1)
        for (int n1 = 0; n1 < R; ++n1) tw[R * B + k2 * R * R + n1 + R * k1] = w((long long)n1 * (k1 + R * k2));
  }
}

inline void build_twiddles(int n, std::vector<float2>& tw) {
  switch (n) {
    case 64: build_twiddles_n<64>(tw); break;
    case 128: build_twiddles_n<128>(tw); break;
    case 256: build_twiddles_n<256>(tw); break;
    case 512: build_twiddles_n<512>(tw); break;
  }
}

#ifdef __CUDACC__
__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }

// Thread -> (line, t) inside a strip.  Row strips: t fastest (a half-warp reads 128 contiguous
// bytes of one row).  Column strips: line fastest (LINES consecutive columns of one row).
template <int N, bool COLS, int LINES_ = FftCfg<N>::LINES>
struct StripThread {
  using S = Strip<N, LINES_>;
  static __device__ __forceinline__ int line() { return COLS ? int(threadIdx.x) % S::LINES : int(threadIdx.x) / S::TPL; }
  static __device__ __forceinline__ int t() { return COLS ? int(threadIdx.x) / S::LINES : int(threadIdx.x) % S::TPL; }
};

// In: v[r] = x[t + TPL r].  Out: v[r] = X[t + TPL r].  `ln` = this thread's line in shared memory.
// Contains barriers: every thread of the CTA must call it.  TW_SMEM: `tw` points to a copy of the
// twiddle table in shared memory (plain loads) instead of global memory (read-only path).
template <int N, bool INV, bool TW_SMEM = false>
__device__ __forceinline__ void fft_regs(float2 (&v)[Strip<N>::R], float2* __restrict__ ln, int t,
                                         const float2* __restrict__ tw) {
  using S = Strip<N>;
  auto twl = [&](int i) { return TW_SMEM ? tw[i] : __ldg(&tw[i]); };
  constexpr int R = S::R, B = S::B, TPL = S::TPL;
  // ---- step 1: DFT_R over n3, twiddle
  RegDft<R, INV>::run(v);
  if (B == 1) {
#pragma unroll
    for (int k1 = 1; k1 < R; ++k1) v[k1] = twmul<INV>(v[k1], twl(k1 * R + t));
  } else {
    const int n2 = t / R;
#pragma unroll
    for (int k1 = 1; k1 < R; ++k1) v[k1] = twmul<INV>(v[k1], twl(k1 * B + n2));
  }
  __syncthreads();                                   // earlier readers of this line are done
#pragma unroll
  for (int k1 = 0; k1 < R; ++k1) ln[pad16(t + TPL * k1)] = v[k1];
  __syncthreads();
  if (B > 1) {
    // ---- step 2: thread q = n1 + R k1 (< R*R): DFT_B over n2 at n1 + R n2 + R B k1, twiddle, in place
    constexpr int PAIRS = R * R;
    if (PAIRS >= TPL || t < PAIRS) {
      const int n1 = t % R, k1 = t / R;
      float2 u[B > 1 ? B : 4];
#pragma unroll
      for (int n2 = 0; n2 < B; ++n2) u[n2] = ln[pad16(n1 + R * n2 + R * B * k1)];
      RegDft<(B > 1 ? B : 4), INV>::run(u);
#pragma unroll
      for (int k2 = 0; k2 < B; ++k2) {
        u[k2] = twmul<INV>(u[k2], twl(R * B + k2 * PAIRS + t));
        ln[pad16(n1 + R * k2 + R * B * k1)] = u[k2];     // same positions this thread read
      }
    }
    __syncthreads();
  }
  // ---- step 3: thread t' = k1 + R k2 reads n1 + R k2 + R B k1 (contiguous in n1), DFT_R over n1
  {
    const int k1 = t % R, k2 = t / R;
    const int base = R * k2 + R * B * k1;
#pragma unroll
    for (int n1 = 0; n1 < R; ++n1) v[n1] = ln[pad16(base + n1)];
    RegDft<R, INV>::run(v);
  }
}
#endif  // __CUDACC__

}  // namespace apic
