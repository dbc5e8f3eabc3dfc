// output.cu - S10 outputs: field on the (uN)^2 grid and the pupil function.
//
// Field (O7 of DESIGN.md): f[X] = sum_k O_hat(k) e^{+2 pi i k.X/(uN)}, X in [0,uN)^2 - the inverse
// DFT of O_hat zero-padded to the uN grid.  With X = u*m + a (a in [0,u)^2) this is u^2 N-point
// inverse transforms of the phase-ramped spectrum O_hat(k) e^{2 pi i k.a/(uN)} (polyphase), so the
// same radix-8/16 line FFT serves 2x and 3x grids.  Rows outside the known region are skipped.
// Pupil: 1[|k|<=R] e^{j phi_hat(k)} on the centred N x N grid.
#include "fft_core.cuh"
#include "plan.hpp"

namespace apic {

__device__ __forceinline__ int wrapNo(int k, int n) { return (k + n) & (n - 1); }

template <int N>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB)
out_rows(DevTables t, const float2* __restrict__ O, float2* __restrict__ TOUT,
         const int32_t* __restrict__ live_count, int chunk0) {
  using S = Strip<N>;
  using TH = StripThread<N, false>;
  extern __shared__ float2 sm[];
  const int slot = blockIdx.z, ax = blockIdx.y;
  if (chunk0 + slot >= *live_count) return;
  const int line = TH::line(), tt = TH::t(), row = blockIdx.x * S::LINES + line;
  const bool valid = row < t.known_nrow;
  const int fy = wrapNo(t.known_row0 + row, N);
  const float2* o = O + size_t(slot) * (N * N) + fy * N;
  const float2* ramp = t.ramp + ax * N;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int fx = tt + S::TPL * r;
    v[r] = valid ? cmul(o[fx], __ldg(&ramp[fx])) : make_float2(0.f, 0.f);
  }
  fft_regs<N, true>(v, sm + line * S::LS, tt, t.tw);
  if (!valid) return;
  const int on = N * t.u;
  float2* to = TOUT + (size_t(slot) * N + fy) * on + ax;
#pragma unroll
  for (int r = 0; r < S::R; ++r) to[(tt + S::TPL * r) * t.u] = v[r];
}

template <int N>
__global__ void __launch_bounds__(Strip<N>::THREADS, Strip<N>::MINB)
out_cols(DevTables t, const float2* __restrict__ TOUT, float2* __restrict__ field,
         const int32_t* __restrict__ live, const int32_t* __restrict__ live_count, int chunk0) {
  using S = Strip<N>;
  using TH = StripThread<N, true>;
  extern __shared__ float2 sm[];
  const int slot = blockIdx.z, ay = blockIdx.y;
  const int tile = resolve_tile_idx(live, live_count, chunk0, slot);
  if (tile < 0) return;
  const int line = TH::line(), tt = TH::t(), x = blockIdx.x * S::LINES + line;
  const int on = N * t.u;
  const float2* to = TOUT + size_t(slot) * N * on + x;
  const float2* ramp = t.ramp + ay * N;
  float2 v[S::R];
#pragma unroll
  for (int r = 0; r < S::R; ++r) {
    const int fy = tt + S::TPL * r;
    const int ky = fy < N / 2 ? fy : fy - N;
    v[r] = (unsigned(ky - t.known_row0) < unsigned(t.known_nrow)) ? cmul(to[size_t(fy) * on], __ldg(&ramp[fy]))
                                                                  : make_float2(0.f, 0.f);
  }
  fft_regs<N, true>(v, sm + line * S::LS, tt, t.tw);
  float2* f = field + size_t(tile) * on * on + x;
#pragma unroll
  for (int r = 0; r < S::R; ++r) f[size_t((tt + S::TPL * r) * t.u + ay) * on] = v[r];
}

__global__ void __launch_bounds__(256) pupil_kernel(DevTables t, const float* __restrict__ coef,
                                                    float2* __restrict__ pupil, const int32_t* __restrict__ live,
                                                    const int32_t* __restrict__ live_count, int chunk0) {
  __shared__ float c_sh[kMaxZern];
  const int slot = blockIdx.y;
  const int tile = resolve_tile_idx(live, live_count, chunk0, slot);
  if (tile < 0) return;
  if (threadIdx.x < t.nz) c_sh[threadIdx.x] = coef[size_t(slot) * t.nz + threadIdx.x];
  __syncthreads();
  const int e = blockIdx.x * 256 + threadIdx.x;
  if (e >= t.n_pupil) return;
  const float* z = t.pupil_zern + size_t(e) * t.nz;
  float phi = 0.f;
  for (int j = 0; j < t.nz; ++j) phi += c_sh[j] * __ldg(&z[j]);
  float sn, cs;
  sincosf(phi, &sn, &cs);
  pupil[size_t(tile) * t.n * t.n + t.pupil_idx[e]] = make_float2(cs, sn);
}

template <int N>
static void output_n(const DevTables& t, const Workspace& w, const LaunchCtx& c, float* d_field) {
  using S = Strip<N>;
  constexpr int TH = S::THREADS, kLines = S::LINES;
  constexpr size_t SM = S::SMEM;
  if (!c.pd->attr_out) {
    cudaFuncSetAttribute(out_rows<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
    cudaFuncSetAttribute(out_cols<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(SM));
    c.pd->attr_out = true;
  }
  dim3 g1((t.known_nrow + kLines - 1) / kLines, t.u, c.chunk_tiles);
  { ProfScope ps(c, CAT_OUT_ROWS);
    out_rows<N><<<g1, TH, SM, c.stream>>>(t, w.O, w.TOUT, c.live_count, c.chunk0); }
  dim3 g2(N * t.u / kLines, t.u, c.chunk_tiles);
  { ProfScope ps(c, CAT_OUT_COLS);
    out_cols<N><<<g2, TH, SM, c.stream>>>(t, w.TOUT, reinterpret_cast<float2*>(d_field), c.live, c.live_count,
                                          c.chunk0); }
}

void launch_output(const DevTables& t, const Workspace& w, const LaunchCtx& c, float* d_field, float* d_pupil) {
  switch (t.n) {
    case 64: output_n<64>(t, w, c, d_field); break;
    case 128: output_n<128>(t, w, c, d_field); break;
    case 256: output_n<256>(t, w, c, d_field); break;
    case 512: output_n<512>(t, w, c, d_field); break;
  }
  if (d_pupil) {
    ProfScope ps(c, CAT_PUPIL);
    pupil_kernel<<<dim3((t.n_pupil + 255) / 256, c.chunk_tiles), 256, 0, c.stream>>>(
        t, w.coef, reinterpret_cast<float2*>(d_pupil), c.live, c.live_count, c.chunk0);
  }
}

}  // namespace apic
