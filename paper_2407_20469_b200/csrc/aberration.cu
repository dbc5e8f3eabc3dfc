// aberration.cu - S6 aberration extraction and S7 correction + stitching.
//
// S6 (Eq. 8-10; readings R8-R12 of DESIGN.md): on every overlap S_il the phase of
// p = S_i conj(S_l) is linear in the pupil phase; in the Noll-Zernike basis (BASELINE.json item 3)
// the rows a(K) are plan-time constants.  The coefficients are found by
//   (i)  a gradient-domain start: rows a(K+e)-a(K), rhs arg(p(K+e) conj p(K)), weights |p(K+e)||p(K)|
//   (ii) refine_iters re-wrapped Gauss-Newton steps c += (A^T W A)^-1 A^T W wrap(beta - A c), W = |p|.
// Each pass forms the augmented Gram matrix [A b 1]^T W [A b 1] as per-CTA partial sums over
// kGramRows rows (deterministic: no atomics), reduced in fp64 and solved by a warp Cholesky.
// S7 (R13, R14): O_hat(k) = mean_i S_i(k) exp(-j[phi(k+kappa_i) - phi(kappa_i)]).
#include "fft_core.cuh"
#include "plan.hpp"

namespace apic {

constexpr float kTwoPi = 6.28318530717958647692f;

__device__ __forceinline__ float wrap_phase(float x) { return x - kTwoPi * rintf(x * (1.f / kTwoPi)); }

// p(K) = S_i(K) conj S_l(K) on every overlap bin (Eq. 9)
__global__ void __launch_bounds__(256) ab_pair_products(DevTables t, const float2* __restrict__ S,
                                                        float2* __restrict__ PR,
                                                        const int32_t* __restrict__ live_count, int chunk0) {
  const int slot = blockIdx.y;
  if (chunk0 + slot >= *live_count) return;
  const int r = blockIdx.x * 256 + threadIdx.x;
  if (r >= t.n_rows) return;
  const float2* s = S + size_t(slot) * t.disc_total;
  const int2 src = reinterpret_cast<const int2*>(t.row_src)[r];
  PR[size_t(slot) * t.n_rows + r] = cmulc(s[src.x], s[src.y]);
}

// MODE 0: gradient rows; MODE 1: full rows with rhs wrap(beta - A c)
template <int MODE>
__global__ void __launch_bounds__(256) ab_gram(DevTables t, const float2* __restrict__ PR,
                                               const float* __restrict__ coef, float* __restrict__ gram,
                                               int gram_parts, int gram_entries,
                                               const int32_t* __restrict__ live_count, int chunk0) {
  extern __shared__ float smf[];
  const int slot = blockIdx.y, part = blockIdx.x;
  if (chunk0 + slot >= *live_count) return;
  const int nz = t.nz, ncol = nz + 2, ld = ncol | 1;
  const int total = MODE == 0 ? t.n_grad : t.n_rows;
  const float2* pr = PR + size_t(slot) * t.n_rows;
  __shared__ float c_sh[kMaxZern];
  if (MODE == 1 && threadIdx.x < nz) c_sh[threadIdx.x] = coef[size_t(slot) * nz + threadIdx.x];
  __syncthreads();
  for (int lr = threadIdx.x; lr < kGramRows; lr += 256) {
    const int r = part * kGramRows + lr;
    float* row = smf + lr * ld;
    if (r >= total) {
      for (int j = 0; j < ncol; ++j) row[j] = 0.f;
      continue;
    }
    float w, b;
    if (MODE == 0) {
      const int2 rr = reinterpret_cast<const int2*>(t.grad_rows)[r];
      const float2 p0 = pr[rr.x], p1 = pr[rr.y];
      const float2 q = cmulc(p1, p0);
      b = atan2f(q.y, q.x);
      w = sqrtf(p0.x * p0.x + p0.y * p0.y) * sqrtf(p1.x * p1.x + p1.y * p1.y);
      const float* a0 = t.a_full + rr.x;
      const float* a1 = t.a_full + rr.y;
      const float sw = sqrtf(w);
      for (int j = 0; j < nz; ++j) row[j] = sw * (__ldg(&a1[size_t(j) * t.n_rows]) - __ldg(&a0[size_t(j) * t.n_rows]));
      row[nz] = sw * b;
      row[nz + 1] = sw;
    } else {
      const float2 p = pr[r];
      const float beta = atan2f(p.y, p.x);
      w = sqrtf(p.x * p.x + p.y * p.y);
      const float* a = t.a_full + r;
      const float sw = sqrtf(w);
      float dot = 0.f;
      for (int j = 0; j < nz; ++j) {
        const float aj = __ldg(&a[size_t(j) * t.n_rows]);
        dot += aj * c_sh[j];
        row[j] = sw * aj;
      }
      b = wrap_phase(beta - dot);                                       // R11
      row[nz] = sw * b;
      row[nz + 1] = sw;
    }
  }
  __syncthreads();
  // Gram entries of the 512 rows: the two halves of the CTA take 256 rows each (four independent accumulators per
  // thread instead of one 512-long dependent chain), the upper half hands its sums over through shared memory.
  float* out = gram + (size_t(slot) * gram_parts + part) * gram_entries;
  float* hand = smf + kGramRows * ld;                    // [gram_entries]
  const int half = threadIdx.x >> 7, r0 = half * (kGramRows / 2);
  for (int e0 = 0; e0 < gram_entries; e0 += 128) {
    const int e = e0 + (threadIdx.x & 127);
    float acc = 0.f;
    if (e < gram_entries) {
      // decode e -> (j <= k) in row-major upper-triangle order
      int j = 0, rem = e;
      while (rem >= ncol - j) { rem -= ncol - j; ++j; }
      const int k = j + rem;
      const float* a = smf + r0 * ld + j;
      const float* b = smf + r0 * ld + k;
      float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll 4
      for (int lr = 0; lr < kGramRows / 2; lr += 4) {
        a0 += a[(lr + 0) * ld] * b[(lr + 0) * ld];
        a1 += a[(lr + 1) * ld] * b[(lr + 1) * ld];
        a2 += a[(lr + 2) * ld] * b[(lr + 2) * ld];
        a3 += a[(lr + 3) * ld] * b[(lr + 3) * ld];
      }
      acc = (a0 + a1) + (a2 + a3);
      if (half) hand[e] = acc;
    }
    __syncthreads();
    if (!half && e < gram_entries) out[e] = acc + hand[e];
  }
}

// One CTA per tile: reduce the partial Grams in fp64, warp Cholesky, update the coefficients.
// MODE 0: c = solve;  MODE 1: c += solve;  MODE 2: no solve, residual RMS -> status, write output.
template <int MODE>
__global__ void __launch_bounds__(128) ab_solve(DevTables t, const float* __restrict__ gram, int gram_parts,
                                                int gram_entries, float* __restrict__ coef,
                                                int32_t* __restrict__ fail, float* __restrict__ d_zernike,
                                                int32_t* __restrict__ d_status, const int32_t* __restrict__ live,
                                                const int32_t* __restrict__ live_count, int chunk0) {
  const int slot = blockIdx.x;
  const int tile = resolve_tile_idx(live, live_count, chunk0, slot);
  if (tile < 0) return;
  const int nz = t.nz, ncol = nz + 2;
  __shared__ double H[(kMaxZern + 2) * (kMaxZern + 2)];
  __shared__ double sol[kMaxZern];
  __shared__ int bad;
  if (threadIdx.x == 0) bad = 0;
  const float* g = gram + size_t(slot) * gram_parts * gram_entries;
  for (int e = threadIdx.x; e < gram_entries; e += 128) {
    double acc = 0.0;
    for (int p = 0; p < gram_parts; ++p) acc += double(g[size_t(p) * gram_entries + e]);
    int j = 0, rem = e;
    while (rem >= ncol - j) { rem -= ncol - j; ++j; }
    const int k = j + rem;
    H[j * ncol + k] = acc;
    H[k * ncol + j] = acc;
  }
  __syncthreads();
  if (MODE == 2) {
    if (threadIdx.x == 0) {
      const double num = H[nz * ncol + nz], den = H[(nz + 1) * ncol + nz + 1];
      const double rms = sqrt(num / den);
      const bool failed = fail[slot] != 0 || !(rms <= 1.0);             // R11: > 1 rad or non-finite
      d_status[tile] = failed ? 3 : 0;
    }
    if (threadIdx.x < nz) d_zernike[size_t(tile) * nz + threadIdx.x] = coef[size_t(slot) * nz + threadIdx.x];
    return;
  }
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    // in-place lower Cholesky of H[0:nz, 0:nz] (column by column)
    for (int k = 0; k < nz; ++k) {
      if (lane == 0) {
        double d = H[k * ncol + k];
        for (int m = 0; m < k; ++m) d -= H[k * ncol + m] * H[k * ncol + m];
        if (!(d > 0.0)) { bad = 1; d = 1.0; }
        H[k * ncol + k] = sqrt(d);
      }
      __syncwarp();
      const double dk = H[k * ncol + k];
      for (int i = k + 1 + lane; i < nz; i += 32) {
        double v = H[i * ncol + k];
        for (int m = 0; m < k; ++m) v -= H[i * ncol + m] * H[k * ncol + m];
        H[i * ncol + k] = v / dk;
      }
      __syncwarp();
    }
    if (lane == 0) {
      // L y = g, L^T x = y with g = column nz of the Gram (A^T W b)
      for (int i = 0; i < nz; ++i) {
        double v = H[nz * ncol + i];                 // row nz was filled symmetrically and is untouched
        for (int m = 0; m < i; ++m) v -= H[i * ncol + m] * sol[m];
        sol[i] = v / H[i * ncol + i];
      }
      for (int i = nz - 1; i >= 0; --i) {
        double v = sol[i];
        for (int m = i + 1; m < nz; ++m) v -= H[m * ncol + i] * sol[m];
        sol[i] = v / H[i * ncol + i];
      }
    }
  }
  __syncthreads();
  if (threadIdx.x < nz) {
    float* c = coef + size_t(slot) * nz;
    const bool ok = (bad == 0) && isfinite(sol[threadIdx.x]);
    if (MODE == 0) c[threadIdx.x] = ok ? float(sol[threadIdx.x]) : 0.f;
    else if (ok) c[threadIdx.x] += float(sol[threadIdx.x]);
  }
  if (threadIdx.x == 0) {
    if (MODE == 0) fail[slot] = bad;
    else if (bad) fail[slot] = 1;
  }
}

// B9: the fit starts from a prior (one per tile) instead of the gradient-domain solve
__global__ void ab_set_init(int nz, const float* __restrict__ init, float* __restrict__ coef, int32_t* __restrict__ fail,
                            const int32_t* __restrict__ live, const int32_t* __restrict__ live_count, int chunk0) {
  const int slot = blockIdx.x;
  const int tile = resolve_tile_idx(live, live_count, chunk0, slot);
  if (tile < 0) return;
  if (threadIdx.x < nz) coef[size_t(slot) * nz + threadIdx.x] = init[size_t(tile) * nz + threadIdx.x];
  if (threadIdx.x == 0) fail[slot] = 0;
}

void launch_aberration(const DevTables& t, const Workspace& w, const LaunchCtx& c, int refine_iters,
                       float* d_zernike, int32_t* d_status, const float* d_init) {
  const size_t sm = (size_t(kGramRows) * ((t.nz + 2) | 1) + size_t(w.gram_entries)) * sizeof(float);
  if (!c.pd->attr_ab) {
    cudaFuncSetAttribute(ab_gram<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(ab_gram<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    c.pd->attr_ab = true;
  }
  dim3 g1((t.n_rows + 255) / 256, c.chunk_tiles);
  { ProfScope ps(c, CAT_AB_PRODUCTS);
    ab_pair_products<<<g1, 256, 0, c.stream>>>(t, w.S, w.PR, c.live_count, c.chunk0); }
  const int parts_g = (t.n_grad + kGramRows - 1) / kGramRows, parts_f = (t.n_rows + kGramRows - 1) / kGramRows;
  if (d_init) {
    ProfScope ps(c, CAT_AB_SOLVE);
    ab_set_init<<<c.chunk_tiles, 64, 0, c.stream>>>(t.nz, d_init, w.coef, w.ab_fail, c.live, c.live_count, c.chunk0);
  } else {
    { ProfScope ps(c, CAT_AB_GRAM);
      ab_gram<0><<<dim3(parts_g, c.chunk_tiles), 256, sm, c.stream>>>(t, w.PR, w.coef, w.gram, parts_g, w.gram_entries,
                                                                        c.live_count, c.chunk0); }
    { ProfScope ps(c, CAT_AB_SOLVE);
      ab_solve<0><<<c.chunk_tiles, 128, 0, c.stream>>>(t, w.gram, parts_g, w.gram_entries, w.coef, w.ab_fail, d_zernike,
                                                       d_status, c.live, c.live_count, c.chunk0); }
  }
  for (int it = 0; it <= refine_iters; ++it) {
    { ProfScope ps(c, CAT_AB_GRAM);
      ab_gram<1><<<dim3(parts_f, c.chunk_tiles), 256, sm, c.stream>>>(t, w.PR, w.coef, w.gram, parts_f,
                                                                        w.gram_entries, c.live_count, c.chunk0); }
    ProfScope ps(c, CAT_AB_SOLVE);
    if (it < refine_iters)
      ab_solve<1><<<c.chunk_tiles, 128, 0, c.stream>>>(t, w.gram, parts_f, w.gram_entries, w.coef, w.ab_fail,
                                                       d_zernike, d_status, c.live, c.live_count, c.chunk0);
    else
      ab_solve<2><<<c.chunk_tiles, 128, 0, c.stream>>>(t, w.gram, parts_f, w.gram_entries, w.coef, w.ab_fail,
                                                       d_zernike, d_status, c.live, c.live_count, c.chunk0);
  }
}

// ---------------------------------------------------------------------------------- S7
__global__ void __launch_bounds__(256) stitch_kernel(DevTables t, const float2* __restrict__ S,
                                                     const float* __restrict__ coef, float2* __restrict__ O,
                                                     const int32_t* __restrict__ live_count, int chunk0) {
  const int slot = blockIdx.y;
  if (chunk0 + slot >= *live_count) return;
  __shared__ float c_sh[kMaxZern];
  if (threadIdx.x < t.nz) c_sh[threadIdx.x] = coef[size_t(slot) * t.nz + threadIdx.x];
  __syncthreads();
  const int b = blockIdx.x * 256 + threadIdx.x;
  if (b >= t.n_union) return;
  const float2* s = S + size_t(slot) * t.disc_total;
  const int e0 = t.union_off[b], e1 = t.union_off[b + 1];
  float2 acc = make_float2(0.f, 0.f);
  for (int q = e0; q < e1; ++q) {
    const int ent = t.union_src[q];
    const float* z = t.disc_zern + size_t(ent) * t.nz;
    float phi = 0.f;
    for (int j = 0; j < t.nz; ++j) phi += c_sh[j] * __ldg(&z[j]);       // phi(k+kappa_i) - phi(kappa_i)
    float sn, cs;
    sincosf(phi, &sn, &cs);
    acc = cadd(acc, cmulc(s[ent], make_float2(cs, sn)));                // * e^{-j phi}
  }
  O[size_t(slot) * t.n * t.n + t.union_f[b]] = cscale(acc, 1.f / float(e1 - e0));
}

void launch_stitch(const DevTables& t, const Workspace& w, const LaunchCtx& c) {
  cudaMemsetAsync(w.O, 0, size_t(c.chunk_tiles) * t.n * t.n * sizeof(float2), c.stream);
  ProfScope ps(c, CAT_STITCH);
  stitch_kernel<<<dim3((t.n_union + 255) / 256, c.chunk_tiles), 256, 0, c.stream>>>(t, w.S, w.coef, w.O, c.live_count,
                                                                                     c.chunk0);
}

}  // namespace apic
