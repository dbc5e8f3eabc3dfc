// reassemble.cu - within-FOV reassembly of overlapping reconstructed tiles.
//
// PAPER.md:171 reconstructs the patches of a field of view one by one "and then stitched together"
// blends overlapping regions "to smoothen any visible seams", proceeding from the top-left corner against what is
// already stitched.  Neither the blend nor the treatment of a complex field's global phase is stated; the readings
// are DESIGN.md B6-B8: regular grid of T x T tiles sharing `overlap` pixels, separable linear blend (weights of the
// covering tiles sum to 1), tiles brought to the global phase of tile (0, 0) in raster order through the correlation
// of their overlaps with the already aligned left / upper neighbour.
//
// Three kernels: (1) the raw overlap correlations C_h, C_v of every tile, all pairs in parallel (they do not depend
// on the factors: sum (u_nb f_nb) conj f = u_nb C), fp64 accumulation in a fixed order; (2) the raster-order scan of
// the unit factors (one thread; a FOV has tens of tiles); (3) the blend, one thread per FOV pixel gathering from the
// <= 4 covering tiles: every tile pixel is read once per pixel it contributes to, the FOV is written once - an HBM
// streaming kernel (bench.py --reassemble reports its GB/s against the measured copy bandwidth).
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "../../include/apic.h"

namespace apic {
void note_cuda_error(cudaError_t e, const char* what);   // api.cu: fills the text apic_last_cuda_error() returns

namespace {

constexpr int kCorrChunks = 16;   // CTAs per (tile, direction): the overlap's lines are dealt round-robin to the chunks

// partial[(tile, dir, chunk)] = sum over the chunk's lines of the overlap with the left (dir 0) / upper (dir 1)
// neighbour of f_nb conj f_tile.  A warp takes a line (a row of the overlap: `ov` pixels for dir 0, T pixels for dir 1),
// fp64 accumulation, fixed order.
__global__ void __launch_bounds__(256) overlap_corr_kernel(const float2* __restrict__ f, int ty, int tx, int T, int ov,
                                                           double2* __restrict__ partial) {
  const int tile = blockIdx.x, dir = blockIdx.y, chunk = blockIdx.z, r = tile / tx, c = tile % tx;
  double re = 0.0, im = 0.0;
  const bool has = dir == 0 ? c > 0 : r > 0;
  if (has) {
    const size_t tt = size_t(T) * T;
    const float2* a = f + size_t(dir == 0 ? tile - 1 : tile - tx) * tt + (dir == 0 ? T - ov : (T - ov) * T);
    const float2* b = f + size_t(tile) * tt;
    const int lines = dir == 0 ? T : ov, len = dir == 0 ? ov : T;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int l = chunk * 8 + warp; l < lines; l += kCorrChunks * 8) {
      const float2* pa = a + size_t(l) * T;
      const float2* pb = b + size_t(l) * T;
      for (int k = lane; k < len; k += 32) {
        const float2 p = __ldg(&pa[k]), q = __ldg(&pb[k]);
        re += double(p.x) * q.x + double(p.y) * q.y;      // p conj q
        im += double(p.y) * q.x - double(p.x) * q.y;
      }
    }
  }
  __shared__ double sre[8], sim[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    re += __shfl_xor_sync(0xffffffffu, re, o);
    im += __shfl_xor_sync(0xffffffffu, im, o);
  }
  if ((threadIdx.x & 31) == 0) { sre[threadIdx.x >> 5] = re; sim[threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double x = 0.0, y = 0.0;
    for (int i = 0; i < 8; ++i) { x += sre[i]; y += sim[i]; }
    partial[(tile * 2 + dir) * kCorrChunks + chunk] = make_double2(x, y);
  }
}

// u(0,0) = 1, u(t) = c / |c| with c = u(left) C_h(t) + u(up) C_v(t), raster order (B8).  All threads first add the
// chunks' partial sums of their correlations in chunk order (into chunk 0's place), then thread 0 scans.
__global__ void __launch_bounds__(256) phase_scan_kernel(double2* __restrict__ partial, int ty, int tx, int align,
                                                         double2* __restrict__ ud, float2* __restrict__ uf) {
  const int n = ty * tx;
  if (align) {
    for (int i = threadIdx.x; i < 2 * n; i += 256) {
      double2 s = make_double2(0.0, 0.0);
      for (int k = 0; k < kCorrChunks; ++k) { s.x += partial[i * kCorrChunks + k].x; s.y += partial[i * kCorrChunks + k].y; }
      partial[i * kCorrChunks] = s;
    }
  }
  __syncthreads();
  if (threadIdx.x != 0) return;
  for (int r = 0; r < ty; ++r)
    for (int c = 0; c < tx; ++c) {
      const int t = r * tx + c;
      double2 u = make_double2(1.0, 0.0);
      if (align && t > 0) {
        double ar = 0.0, ai = 0.0;
        if (c > 0) {
          const double2 un = ud[t - 1], k = partial[(t * 2) * kCorrChunks];
          ar += un.x * k.x - un.y * k.y;
          ai += un.x * k.y + un.y * k.x;
        }
        if (r > 0) {
          const double2 un = ud[t - tx], k = partial[(t * 2 + 1) * kCorrChunks];
          ar += un.x * k.x - un.y * k.y;
          ai += un.x * k.y + un.y * k.x;
        }
        const double m = sqrt(ar * ar + ai * ai);
        if (m > 0.0) u = make_double2(ar / m, ai / m);
      }
      ud[t] = u;
      uf[t] = make_float2(float(u.x), float(u.y));
    }
}

// 1-D blend weight of pixel i of tile idx (of n) along one axis (B7)
__device__ __forceinline__ float ramp(int i, int idx, int n, int T, int ov, float inv_ov) {
  if (idx > 0 && i < ov) return (float(i) + 0.5f) * inv_ov;
  if (idx < n - 1 && i >= T - ov) return 1.f - (float(i - (T - ov)) + 0.5f) * inv_ov;
  return 1.f;
}

// PX = 2: two neighbouring pixels per thread with 16-byte accesses (T, overlap and W even: the pair then lies in the
// same tile column and on the same side of every overlap boundary); PX = 1: any geometry.
template <int PX>
__global__ void __launch_bounds__(256) blend_kernel(const float2* __restrict__ f, const float2* __restrict__ u, int ty, int tx,
                                                    int T, int ov, int H, int W, float2* __restrict__ out) {
  const int X = (blockIdx.x * 256 + threadIdx.x) * PX;
  if (X >= W) return;
  const int step = T - ov;
  const float inv_ov = ov > 0 ? 1.f / float(ov) : 0.f;
  const int c1 = min(X / step, tx - 1), x1 = X - c1 * step;
  const bool left = c1 > 0 && x1 < ov;
  float wx[PX];
#pragma unroll
  for (int p = 0; p < PX; ++p) wx[p] = ramp(x1 + p, c1, tx, T, ov, inv_ov);
  const size_t tt = size_t(T) * T;
  for (int Y = blockIdx.y; Y < H; Y += gridDim.y) {
    const int r1 = min(Y / step, ty - 1), y1 = Y - r1 * step;
    const bool up = r1 > 0 && y1 < ov;
    const float wy1 = ramp(y1, r1, ty, T, ov, inv_ov);
    float2 acc[PX];
#pragma unroll
    for (int p = 0; p < PX; ++p) acc[p] = make_float2(0.f, 0.f);
    auto add = [&](int r, int c, int y, int x, float wy, bool other_x) {
      const float2* src = f + size_t(r * tx + c) * tt + size_t(y) * T + x;
      const float2 q = __ldg(&u[r * tx + c]);
      float2 v[PX];
      if (PX == 2) {
        const float4 t4 = __ldg(reinterpret_cast<const float4*>(src));
        v[0] = make_float2(t4.x, t4.y);
        v[PX - 1] = make_float2(t4.z, t4.w);
      } else {
        v[0] = __ldg(src);
      }
#pragma unroll
      for (int p = 0; p < PX; ++p) {
        const float w = wy * (other_x ? 1.f - wx[p] : wx[p]);
        acc[p].x += w * (q.x * v[p].x - q.y * v[p].y);
        acc[p].y += w * (q.x * v[p].y + q.y * v[p].x);
      }
    };
    add(r1, c1, y1, x1, wy1, false);
    if (left) add(r1, c1 - 1, y1, x1 + step, wy1, true);
    if (up) add(r1 - 1, c1, y1 + step, x1, 1.f - wy1, false);
    if (up && left) add(r1 - 1, c1 - 1, y1 + step, x1 + step, 1.f - wy1, true);
    float2* dst = out + size_t(Y) * W + X;
    if (PX == 2) *reinterpret_cast<float4*>(dst) = make_float4(acc[0].x, acc[0].y, acc[PX - 1].x, acc[PX - 1].y);
    else *dst = acc[0];
  }
}

}  // namespace
}  // namespace apic

extern "C" {

size_t apic_reassemble_work_bytes(int tiles_y, int tiles_x) {
  if (tiles_y < 1 || tiles_x < 1) return 0;
  return size_t(tiles_y) * tiles_x * (2 * apic::kCorrChunks + 1) * sizeof(double2);   // partial C_h, C_v; the fp64 factors
}

int apic_reassemble(const float* d_fields, int tiles_y, int tiles_x, int tile_px, int overlap, int align, float* d_fov,
                    float* d_factors, void* d_work, void* cuda_stream) {
  using namespace apic;
  if (!d_fields || !d_fov || !d_factors || !d_work) return APIC_EINVAL;
  if (tiles_y < 1 || tiles_x < 1 || tile_px < 1 || overlap < 0 || 2 * overlap > tile_px) return APIC_EINVAL;
  if (size_t(tiles_y) * tiles_x > 65535u) return APIC_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int n = tiles_y * tiles_x, T = tile_px, step = T - overlap;
  const int H = tiles_y * step + overlap, W = tiles_x * step + overlap;
  double2* corr = static_cast<double2*>(d_work);
  double2* ud = corr + size_t(n) * 2 * kCorrChunks;
  const float2* f = reinterpret_cast<const float2*>(d_fields);
  cudaGetLastError();
  if (align && overlap > 0) overlap_corr_kernel<<<dim3(n, 2, kCorrChunks), 256, 0, s>>>(f, tiles_y, tiles_x, T, overlap, corr);
  phase_scan_kernel<<<1, 256, 0, s>>>(corr, tiles_y, tiles_x, align && overlap > 0, ud, reinterpret_cast<float2*>(d_factors));
  const bool vec = (T % 2 == 0) && (overlap % 2 == 0) && (reinterpret_cast<uintptr_t>(d_fields) % 16 == 0) &&
                   (reinterpret_cast<uintptr_t>(d_fov) % 16 == 0);          // then W is even too
  const int gy = H < 65535 ? H : 65535;
  if (vec)
    blend_kernel<2><<<dim3((W / 2 + 255) / 256, gy), 256, 0, s>>>(f, reinterpret_cast<const float2*>(d_factors), tiles_y, tiles_x,
                                                                 T, overlap, H, W, reinterpret_cast<float2*>(d_fov));
  else
    blend_kernel<1><<<dim3((W + 255) / 256, gy), 256, 0, s>>>(f, reinterpret_cast<const float2*>(d_factors), tiles_y, tiles_x, T,
                                                             overlap, H, W, reinterpret_cast<float2*>(d_fov));
  return cudaGetLastError() == cudaSuccess ? APIC_OK : APIC_ECUDA;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// apic_reassemble_static: the same three kernels, for callers that have no way to hand over a d_work buffer.
//
// Who that is: code that runs where device memory can no longer be requested - a reassembly step that sits inside a
// host application whose memory was handed out in full at start-up (an acquisition loop with a fixed arena, a plugin
// whose host owns the allocator), or a latency-bound loop in which a cudaMalloc would stall every stream of the
// process.  For them the correlation partial sums and the fp64 unit factors live in an array that is part of the
// library image itself: it exists on a GPU from the moment the library's device code is loaded there and until the
// process exits, whether or not it is ever used, so its size is a hard limit, kept modest.
//
// `g_reassemble_scratch` below is, on the host side of this file, only a handle that the CUDA runtime knows how to
// look up.  It is NOT the device address (a kernel that were passed `g_reassemble_scratch` from host code would read
// some host location, or fault); the device address is asked for once per device with cudaGetSymbolAddress while that
// device is current, and that address is what the kernels get.
// ---------------------------------------------------------------------------------------------------------------------
#define APIC_REASSEMBLE_STATIC_MAX_TILES 1024   /* 1024 x (2 x 16 + 1) x 16 B = 528 KiB on every GPU that loads libapic */

static __device__ __align__(256) double2 g_reassemble_scratch[size_t(APIC_REASSEMBLE_STATIC_MAX_TILES) *
                                                              (2 * apic::kCorrChunks + 1)];

namespace apic {
namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
double2* g_static_scratch_of_device[kStaticMaxDevices] = {};   // device address of g_reassemble_scratch, per device

// Device address of the scratch on the CURRENT device (looked up at the first call on that device, then cached).
int static_scratch(double2** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { note_cuda_error(e, "apic_reassemble_static: cudaGetDevice"); return APIC_ECUDA; }
  if (dev < 0 || dev >= kStaticMaxDevices) return APIC_EINVAL;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_scratch_of_device[dev]) {
    double2* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_reassemble_scratch);
    if (e != cudaSuccess || !p) {
      note_cuda_error(e, "apic_reassemble_static: cudaGetSymbolAddress(g_reassemble_scratch)");
      return APIC_ECUDA;
    }
    g_static_scratch_of_device[dev] = p;
  }
  *out = g_static_scratch_of_device[dev];
  return APIC_OK;
}

}  // namespace
}  // namespace apic

extern "C" {

int apic_reassemble_static_max_tiles(void) { return APIC_REASSEMBLE_STATIC_MAX_TILES; }

int apic_reassemble_static(const float* d_fields, int tiles_y, int tiles_x, int tile_px, int overlap, int align,
                           float* d_fov, float* d_factors, void* cuda_stream) {
  if (tiles_y < 1 || tiles_x < 1) return APIC_EINVAL;
  if (size_t(tiles_y) * size_t(tiles_x) > size_t(APIC_REASSEMBLE_STATIC_MAX_TILES)) return APIC_ESCRATCH;
  double2* work = nullptr;
  const int rc = apic::static_scratch(&work);
  if (rc != APIC_OK) return rc;
  // Nothing in the scratch has to start at zero: overlap_corr_kernel stores every partial sum that phase_scan_kernel
  // adds up (a zero where a tile has no left / upper neighbour), and the scan writes each factor before it reads it.
  // What an earlier call left behind is therefore never looked at, and no clearing pass is enqueued.
  return apic_reassemble(d_fields, tiles_y, tiles_x, tile_px, overlap, align, d_fov, d_factors, work, cuda_stream);
}

}  // extern "C"
