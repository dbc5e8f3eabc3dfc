// fft_core.cuh - batched shared-memory complex FFT building blocks (libapic kernel K1).
//
// Every transform of the APIC path (Eq. 5-7; Eq. 13 mat-vecs) is a
// 2-D DFT of an N x N tile, N in {64,128,256,512}.  It is executed as 1-D "line" transforms over
// strips of kLines lines held in shared memory: a row strip (lines = consecutive rows) or a column
// strip (lines = consecutive columns, 128-byte global segments per row).  A line transform is a
// Stockham autosort FFT with register-resident radix-8/16 butterflies (two or three passes through
// shared memory), natural order in and out, unnormalised:
//     forward  X[k] = sum_n x[n] e^{-2 pi i k n / N},    inverse  x[n] = sum_k X[k] e^{+2 pi i k n / N}.
// Twiddles come from an fp64-computed table tw[m] = e^{-2 pi i m / N} (plan-time).
#pragma once
#include <cuda_runtime.h>

namespace apic {

constexpr int kLines = 16;  // lines per strip: 16 complex64 = one 128-byte global segment per row

__host__ __device__ constexpr int line_stride(int n) { return n + n / 16 + 1; }  // odd-ish, padded
__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }
__host__ __device__ constexpr size_t strip_smem_bytes(int n) { return size_t(kLines) * line_stride(n) * sizeof(float2); }

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {  // a * conj(b)
  return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ float2 cscale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }

// multiply by e^{-+ i pi/2}: forward (-i), inverse (+i)
template <bool INV>
__device__ __forceinline__ float2 rot90(float2 a) {
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}
// multiply by (c - i s) forward, (c + i s) inverse
template <bool INV>
__device__ __forceinline__ float2 rot(float2 a, float c, float s) {
  return INV ? make_float2(a.x * c - a.y * s, a.y * c + a.x * s)
             : make_float2(a.x * c + a.y * s, a.y * c - a.x * s);
}

// ---- register DFTs, natural order in/out: V[m] = sum_r v[r] e^{-+ 2 pi i r m / R}
template <bool INV>
__device__ __forceinline__ void dft4(float2& a, float2& b, float2& c, float2& d) {
  float2 t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = rot90<INV>(csub(b, d));
  a = cadd(t0, t2);
  b = cadd(t1, t3);
  c = csub(t0, t2);
  d = csub(t1, t3);
}

template <int R, bool INV>
struct RegDft;

template <bool INV>
struct RegDft<2, INV> {
  static __device__ __forceinline__ void run(float2 (&v)[2]) {
    float2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  }
};

template <bool INV>
struct RegDft<4, INV> {
  static __device__ __forceinline__ void run(float2 (&v)[4]) { dft4<INV>(v[0], v[1], v[2], v[3]); }
};

template <bool INV>
struct RegDft<8, INV> {
  static __device__ __forceinline__ void run(float2 (&v)[8]) {
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
  static __device__ __forceinline__ void run(float2 (&v)[16]) {
    constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;  // pi/8
    constexpr float h = 0.70710678118654752440f;
    // X_b[m1] = DFT4 over a of v[4a+b]
    float2 x[4][4];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      x[b][0] = v[b]; x[b][1] = v[4 + b]; x[b][2] = v[8 + b]; x[b][3] = v[12 + b];
      dft4<INV>(x[b][0], x[b][1], x[b][2], x[b][3]);
    }
    // twiddle w16^{b*m1}
    x[1][1] = rot<INV>(x[1][1], c1, s1);   // e=1
    x[1][2] = rot<INV>(x[1][2], h, h);     // e=2
    x[1][3] = rot<INV>(x[1][3], s1, c1);   // e=3
    x[2][1] = rot<INV>(x[2][1], h, h);     // e=2
    x[2][2] = rot90<INV>(x[2][2]);         // e=4
    x[2][3] = rot<INV>(x[2][3], -h, h);    // e=6
    x[3][1] = rot<INV>(x[3][1], s1, c1);   // e=3
    x[3][2] = rot<INV>(x[3][2], -h, h);    // e=6
    x[3][3] = rot<INV>(x[3][3], -c1, -s1); // e=9: cos(9pi/8) = -c1, sin(9pi/8) = -s1
    // V[m1 + 4 m2] = DFT4 over b of X_b[m1]
#pragma unroll
    for (int m1 = 0; m1 < 4; ++m1) {
      float2 y0 = x[0][m1], y1 = x[1][m1], y2 = x[2][m1], y3 = x[3][m1];
      dft4<INV>(y0, y1, y2, y3);
      v[m1] = y0; v[m1 + 4] = y1; v[m1 + 8] = y2; v[m1 + 12] = y3;
    }
  }
};

// ---- per-N factorisation
template <int N> struct FftCfg;
// MINB = CTAs per SM the strip kernels are compiled for (register cap = 64K / (THREADS * MINB))
template <> struct FftCfg<64>  { static constexpr int R1 = 8,  R2 = 8,  R3 = 1, THREADS = 128, MINB = 8; };
template <> struct FftCfg<128> { static constexpr int R1 = 16, R2 = 8,  R3 = 1, THREADS = 128, MINB = 8; };
template <> struct FftCfg<256> { static constexpr int R1 = 16, R2 = 16, R3 = 1, THREADS = 256, MINB = 4; };
template <> struct FftCfg<512> { static constexpr int R1 = 8,  R2 = 8,  R3 = 8, THREADS = 512, MINB = 1; };

// One Stockham pass over all kLines lines of the strip, in place (read all -> sync -> write all).
template <int N, int R, int NS, bool INV>
__device__ __forceinline__ void stockham_pass(float2* __restrict__ sm, const float2* __restrict__ tw) {
  constexpr int THREADS = FftCfg<N>::THREADS;
  constexpr int NB = N / R;               // butterflies per line
  constexpr int TOTAL = kLines * NB;
  static_assert(TOTAL % THREADS == 0, "strip does not divide over the block");
  constexpr int BPT = TOTAL / THREADS;
  constexpr int LS = line_stride(N);
  float2 v[BPT][R];
#pragma unroll
  for (int b = 0; b < BPT; ++b) {
    const int g = threadIdx.x + b * THREADS;
    const int line = g / NB, j = g % NB;
    const float2* L = sm + line * LS;
#pragma unroll
    for (int r = 0; r < R; ++r) v[b][r] = L[pad16(j + r * NB)];
    if (NS > 1) {
      const int k = j & (NS - 1);
      constexpr int STEP = N / (NS * R);
#pragma unroll
      for (int r = 1; r < R; ++r) {
        float2 w = __ldg(&tw[r * k * STEP]);
        if (INV) w.y = -w.y;
        v[b][r] = cmul(v[b][r], w);
      }
    }
    RegDft<R, INV>::run(v[b]);
  }
  __syncthreads();
#pragma unroll
  for (int b = 0; b < BPT; ++b) {
    const int g = threadIdx.x + b * THREADS;
    const int line = g / NB, j = g % NB;
    const int k = j & (NS - 1);
    const int j0 = (j - k) * R + k;
    float2* L = sm + line * LS;
#pragma unroll
    for (int m = 0; m < R; ++m) L[pad16(j0 + m * NS)] = v[b][m];
  }
  __syncthreads();
}

// Transforms every line of the strip in place.  Caller must __syncthreads() after filling sm.
template <int N, bool INV>
__device__ __forceinline__ void fft_lines(float2* __restrict__ sm, const float2* __restrict__ tw) {
  using C = FftCfg<N>;
  stockham_pass<N, C::R1, 1, INV>(sm, tw);
  stockham_pass<N, C::R2, C::R1, INV>(sm, tw);
  if constexpr (C::R3 > 1) stockham_pass<N, C::R3, C::R1 * C::R2, INV>(sm, tw);
}

// element (line l, position e) of the strip
template <int N>
__device__ __forceinline__ float2& strip_at(float2* sm, int l, int e) {
  return sm[l * line_stride(N) + pad16(e)];
}

// ---- strip <-> global helpers.  Row strip: line l = row (row index given per line by the caller),
// position = x.  Column strip: line l = column x0 + l, position = row.
// Loop shapes: row strips iterate idx -> (l = idx / N, e = idx % N)  (coalesced along x);
//              column strips iterate idx -> (l = idx % kLines, e = idx / kLines) (128 B per row).

template <int N>
__device__ __forceinline__ void strip_zero(float2* sm) {
  for (int idx = threadIdx.x; idx < kLines * line_stride(N); idx += FftCfg<N>::THREADS)
    sm[idx] = make_float2(0.f, 0.f);
}

}  // namespace apic
