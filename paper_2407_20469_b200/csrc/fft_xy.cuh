// fft_xy.cuh - mixed-radix line FFT of length L = 16 * R1, R1 in {6, 8, 10, 12, 16}
// (L = 96, 128, 160, 192, 256), used by the darkfield solver on its reduced cyclic grids
// (df_mgrid.cu; Eq. 13 mat-vecs).
//
// A strip holds 16 lines and is worked on by 256 threads.  Two mirrored transform types move the
// data between two register distributions with ONE shared-memory exchange and ONE barrier each:
//
//   layout A ("16 x R1"):  thread t  (t < 16)   holds  x[t  + 16 r],  r  < R1
//   layout B ("R1 x 16"):  thread k1 (k1 < R1)  holds  x[k1 + R1 k2], k2 < 16
//
//   type X : A -> B     DFT_R1 over r, twiddle W_L^{t k1}, exchange, DFT_16 over t
//   type Y : B -> A     DFT_16 over k2, twiddle W_L^{k1 k'}, exchange, DFT_R1 over k1
//
// so that "X, pointwise, Y" (IFFT . multiply . FFT) chains through registers, and both layouts
// give coalesced global accesses (consecutive threads <-> consecutive elements).  Natural order in
// and out, unnormalised, forward = e^{-2 pi i k n / L}.  DFT_6/10/12 are prime-factor (Good-Thomas)
// compositions of DFT_2/3/4/5: no internal twiddles.
#pragma once
#include "fft_core.cuh"

namespace apic {

// ---- small register DFTs (natural order in/out)
template <bool INV>
__host__ __device__ __forceinline__ void dft2(float2& a, float2& b) {
  const float2 t = csub(a, b);
  a = cadd(a, b);
  b = t;
}
template <bool INV>
__host__ __device__ __forceinline__ void dft3(float2& a, float2& b, float2& c) {
  constexpr float s3 = 0.86602540378443864676f;
  const float2 s = cadd(b, c), d = csub(b, c);
  const float2 m = make_float2(a.x - 0.5f * s.x, a.y - 0.5f * s.y);
  a = cadd(a, s);
  // forward: X1 = m - i s3 d, X2 = m + i s3 d ; inverse: swapped
  const float2 r = INV ? make_float2(-s3 * d.y, s3 * d.x) : make_float2(s3 * d.y, -s3 * d.x);
  b = cadd(m, r);
  c = csub(m, r);
}
template <bool INV>
__host__ __device__ __forceinline__ void dft5(float2& a, float2& b, float2& c, float2& d, float2& e) {
  constexpr float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;   // cos 72, cos 144
  constexpr float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;    // sin 72, sin 144
  const float2 p1 = cadd(b, e), p2 = cadd(c, d), m1 = csub(b, e), m2 = csub(c, d);
  const float2 a1 = make_float2(a.x + c1 * p1.x + c2 * p2.x, a.y + c1 * p1.y + c2 * p2.y);
  const float2 a2 = make_float2(a.x + c2 * p1.x + c1 * p2.x, a.y + c2 * p1.y + c1 * p2.y);
  const float2 t1 = make_float2(s1 * m1.x + s2 * m2.x, s1 * m1.y + s2 * m2.y);
  const float2 t2 = make_float2(s2 * m1.x - s1 * m2.x, s2 * m1.y - s1 * m2.y);
  a = cadd(a, cadd(p1, p2));
  // forward: X1 = a1 - i t1, X4 = a1 + i t1, X2 = a2 - i t2, X3 = a2 + i t2
  const float2 r1 = INV ? make_float2(-t1.y, t1.x) : make_float2(t1.y, -t1.x);
  const float2 r2 = INV ? make_float2(-t2.y, t2.x) : make_float2(t2.y, -t2.x);
  b = cadd(a1, r1);
  e = csub(a1, r1);
  c = cadd(a2, r2);
  d = csub(a2, r2);
}

// Prime-factor DFT of length N1*N2 (coprime): n = (N2 n1 + N1 n2) mod N, k = (A k1 + B k2) mod N with
// A = N2 (N2^-1 mod N1), B = N1 (N1^-1 mod N2).
template <bool INV>
struct RegDft<6, INV> {     // 3 x 2: n = 2 n1 + 3 n2, k = 4 k1 + 3 k2
  static __host__ __device__ __forceinline__ void run(float2 (&v)[6]) {
    float2 x[2][3];
#pragma unroll
    for (int n2 = 0; n2 < 2; ++n2) {
#pragma unroll
      for (int n1 = 0; n1 < 3; ++n1) x[n2][n1] = v[(2 * n1 + 3 * n2) % 6];
      dft3<INV>(x[n2][0], x[n2][1], x[n2][2]);
    }
#pragma unroll
    for (int k1 = 0; k1 < 3; ++k1) {
      dft2<INV>(x[0][k1], x[1][k1]);
      v[(4 * k1) % 6] = x[0][k1];
      v[(4 * k1 + 3) % 6] = x[1][k1];
    }
  }
};
template <bool INV>
struct RegDft<10, INV> {    // 5 x 2: n = 2 n1 + 5 n2, k = 6 k1 + 5 k2
  static __host__ __device__ __forceinline__ void run(float2 (&v)[10]) {
    float2 x[2][5];
#pragma unroll
    for (int n2 = 0; n2 < 2; ++n2) {
#pragma unroll
      for (int n1 = 0; n1 < 5; ++n1) x[n2][n1] = v[(2 * n1 + 5 * n2) % 10];
      dft5<INV>(x[n2][0], x[n2][1], x[n2][2], x[n2][3], x[n2][4]);
    }
#pragma unroll
    for (int k1 = 0; k1 < 5; ++k1) {
      dft2<INV>(x[0][k1], x[1][k1]);
      v[(6 * k1) % 10] = x[0][k1];
      v[(6 * k1 + 5) % 10] = x[1][k1];
    }
  }
};
template <bool INV>
struct RegDft<12, INV> {    // 3 x 4: n = 4 n1 + 3 n2, k = 4 k1 + 9 k2
  static __host__ __device__ __forceinline__ void run(float2 (&v)[12]) {
    float2 x[4][3];
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) {
#pragma unroll
      for (int n1 = 0; n1 < 3; ++n1) x[n2][n1] = v[(4 * n1 + 3 * n2) % 12];
      dft3<INV>(x[n2][0], x[n2][1], x[n2][2]);
    }
#pragma unroll
    for (int k1 = 0; k1 < 3; ++k1) {
      dft4<INV>(x[0][k1], x[1][k1], x[2][k1], x[3][k1]);
#pragma unroll
      for (int k2 = 0; k2 < 4; ++k2) v[(4 * k1 + 9 * k2) % 12] = x[k2][k1];
    }
  }
};

// Host: twiddles of the X/Y exchange, tw[a * 16 + b] = e^{-2 pi i a b / L}, a, b < 16 (L = 16 R1): a symmetric
// table, read as tw[k1 * 16 + t] by type X and as tw[k' * 16 + k1] by type Y, so that in both the threads of a
// warp (consecutive t, or consecutive k1) read consecutive entries.  For R1 = 16 this is the table of
// fft_core.cuh's N = 256 transform.
inline void build_twiddles_xy(int r1, std::vector<float2>& tw) {
  const int L = 16 * r1;
  tw.assign(256, make_float2(1.f, 0.f));
  for (int k1 = 0; k1 < 16; ++k1)
    for (int t = 0; t < 16; ++t) {
      const double a = -2.0 * M_PI * double((t * k1) % L) / double(L);
      tw[k1 * 16 + t] = make_float2(float(std::cos(a)), float(std::sin(a)));
    }
}
constexpr int kXyBuf = 4608;     // float2 entries of one exchange buffer (max over layouts: 16*16*18)

#ifdef __CUDACC__
// Thread roles inside a 256-thread strip of 16 lines.
//   COLS (lines = 16 consecutive columns): line = tid % 16 in both layouts, t / k1 = tid / 16
//        (threads with k1 >= R1 idle in layout B: whole warps).
//   ROWS (lines = 16 rows): layout A line = tid / 16, t = tid % 16 (a half-warp reads 128 contiguous
//        bytes of its row); layout B compact: q = tid < 16 R1, line = q / R1, k1 = q % R1.
template <int R1, bool COLS>
struct XY {
  static __device__ __forceinline__ int a_line() { return COLS ? int(threadIdx.x) & 15 : int(threadIdx.x) >> 4; }
  static __device__ __forceinline__ int a_t() { return COLS ? int(threadIdx.x) >> 4 : int(threadIdx.x) & 15; }
  static __device__ __forceinline__ bool b_active() { return COLS ? (int(threadIdx.x) >> 4) < R1 : int(threadIdx.x) < 16 * R1; }
  static __device__ __forceinline__ int b_line() { return COLS ? int(threadIdx.x) & 15 : int(threadIdx.x) / R1; }
  static __device__ __forceinline__ int b_k1() { return COLS ? int(threadIdx.x) >> 4 : int(threadIdx.x) % R1; }
  // row layouts in shared memory: X exchange [line][k1][t] with k1-stride 18; Y exchange [line][k'][k1] with k'-stride R1P
  static constexpr int R1P = (R1 == 6) ? 6 : (R1 == 8 || R1 == 10) ? 10 : (R1 == 12) ? 14 : 18;
  // line stride of the Y exchange: consecutive lines shifted by R1 entries in bank space, so that the
  // compact layout-B warps (32 / R1 lines each) write conflict-free
  static constexpr int LSY = 16 * R1P + (R1 % 16);
};

// Type X: in  v[r] = x[t + 16 r], r < R1 (layout A);  out v[k2] = X[k1 + R1 k2], k2 < 16 (layout B, active threads only).
// One barrier; `buf` must not be read by any thread after the caller's previous barrier.
template <int R1, bool INV, bool COLS>
__device__ __forceinline__ void fft_x(float2 (&v)[16], float2* __restrict__ buf, const float2* __restrict__ tw) {
  using M = XY<R1, COLS>;
  {
    float2 a[R1];
#pragma unroll
    for (int r = 0; r < R1; ++r) a[r] = v[r];
    RegDft<R1, INV>::run(a);
    const int line = M::a_line(), t = M::a_t();
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) {
      const float2 y = k1 ? twmul<INV>(a[k1], tw[k1 * 16 + t]) : a[0];
      if (COLS) buf[(k1 * 16 + t) * 16 + line] = y;
      else buf[line * (R1 * 18) + k1 * 18 + t] = y;
    }
  }
  __syncthreads();
  if (M::b_active()) {
    const int line = M::b_line(), k1 = M::b_k1();
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

// Type Y: in  v[k2] = x[k1 + R1 k2], k2 < 16 (layout B);  out v[r] = X[t + 16 r], r < R1 (layout A).
template <int R1, bool INV, bool COLS>
__device__ __forceinline__ void fft_y(float2 (&v)[16], float2* __restrict__ buf, const float2* __restrict__ tw) {
  using M = XY<R1, COLS>;
  if (M::b_active()) {
    const int line = M::b_line(), k1 = M::b_k1();
    RegDft<16, INV>::run(v);
#pragma unroll
    for (int kp = 0; kp < 16; ++kp) {
      const float2 y = kp ? twmul<INV>(v[kp], tw[kp * 16 + k1]) : v[0];
      if (COLS) buf[(kp * R1 + k1) * 16 + line] = y;
      else buf[line * M::LSY + kp * M::R1P + k1] = y;
    }
  }
  __syncthreads();
  {
    const int line = M::a_line(), kp = M::a_t();
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
#endif  // __CUDACC__

}  // namespace apic
