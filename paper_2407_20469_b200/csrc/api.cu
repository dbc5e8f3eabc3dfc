// api.cu - the C ABI of libapic (include/apic.h): plan construction (host fp64 geometry ->
// device tables + workspace) and the enqueue order of the hot path.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/apic.h"
#include "fft_core.cuh"
#include "fft_xy.cuh"
#include "plan.hpp"

using namespace apic;

namespace {

thread_local std::string g_cuda_err;
thread_local std::string g_plan_err;

bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  g_cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
  return false;
}

}  // namespace

namespace apic {
// for the translation units that have no plan (reassemble.cu): same text slot as cuda_ok()
void note_cuda_error(cudaError_t e, const char* what) { cuda_ok(e == cudaSuccess ? cudaErrorUnknown : e, what); }
}  // namespace apic

// One workspace set: everything a pass of apic_reconstruct writes.  The plan owns two; the second is
// allocated on first use by apic_reconstruct_host so that the kernels of one sub-batch run beside the
// copies (and the kernels) of its neighbours.
struct WsSet {
  Workspace ws{};
  BatchState bs{};
  int32_t* h_live_count = nullptr;   // pinned
  bool ready = false;
  cudaStream_t aux = nullptr;        // KK sub-passes alternate between the caller's stream and this one
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
};

struct apic_plan {
  apic_params params{};
  HostTables host;
  DevTables dev{};
  PlanDevice pd{};
  std::vector<DarkDev> dark;
  const DarkDev* d_dark = nullptr;   // device copy of `dark`
  WsSet set[2];
  int chunk = 1, max_unknown = 1;
  std::vector<void*> allocs;
  size_t table_bytes = 0, workspace_bytes = 0;
  int launches = 0;
  Profiler prof;
  // staging buffers of apic_reconstruct_host (grow-only)
  float *st_int = nullptr, *st_field = nullptr, *st_zern = nullptr, *st_pupil = nullptr;
  int32_t* st_status = nullptr;
  int st_batch = 0;
  bool st_has_pupil = false;
  uint16_t* st_raw = nullptr;        // staging of apic_reconstruct_host_u16
  float* st_scale = nullptr;
  int st_raw_batch = 0, st_int_batch = 0;
  // apic_submit_host / apic_wait_host: one pipeline slot per workspace set
  struct HostSlot {
    float* in_f32 = nullptr;
    uint16_t* in_u16 = nullptr;
    float* in_scale = nullptr;
    float *field = nullptr, *zern = nullptr, *pupil = nullptr;
    int32_t* status = nullptr;
    int cap_f32 = 0, cap_u16 = 0, cap_out = 0;
    bool has_pupil = false, busy = false;
    int rc = 0;
    cudaStream_t ks = nullptr;
    cudaEvent_t in_done = nullptr, k_done = nullptr, out_done = nullptr;
  } slot[2];
  // apic_reconstruct_host: copy streams, a second compute stream and per-part events (upload done, kernels done)
  static constexpr int kMaxParts = 8;
  cudaStream_t copy_in = nullptr, copy_out = nullptr, aux = nullptr;
  cudaEvent_t part_ev[2 * kMaxParts + 2] = {};

  template <class T>
  bool dalloc(T** p, size_t count, bool table) {
    void* q = nullptr;
    const size_t bytes = (count ? count : 1) * sizeof(T);
    if (!cuda_ok(cudaMalloc(&q, bytes), "cudaMalloc")) return false;
    allocs.push_back(q);
    (table ? table_bytes : workspace_bytes) += bytes;
    *p = static_cast<T*>(q);
    return true;
  }
  template <class T>
  bool upload(const T** p, const std::vector<T>& v) {
    T* q = nullptr;
    if (!dalloc(&q, v.size(), true)) return false;
    if (!v.empty() && !cuda_ok(cudaMemcpy(q, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice), "cudaMemcpy"))
      return false;
    *p = q;
    return true;
  }
  bool alloc_set(WsSet& z);
};

bool apic_plan::alloc_set(WsSet& z) {
  if (z.ready) return true;
  Workspace& w = z.ws;
  const HostTables& h = host;
  const DevTables& d = dev;
  const size_t nn = size_t(h.n) * h.n, c = size_t(chunk);
  const int nz = h.nz;
  w.chunk = chunk;
  w.max_unknown = max_unknown;
  const int ncol = nz + 2;
  w.gram_entries = ncol * (ncol + 1) / 2;
  w.gram_parts = (std::max(d.n_rows, d.n_grad) + kGramRows - 1) / kGramRows;
  const size_t n_led = std::max<size_t>(1, h.dark.size());
  bool ok = true;
  const size_t first_alloc = allocs.size(), bytes_before = workspace_bytes;
  ok = ok && dalloc(&w.G, c * h.nb * size_t(h.kk_n) * h.kk_n, false);
  w.KP = nullptr;
  if (h.kk_n != h.n) ok = ok && dalloc(&w.KP, c * h.nb * nn, false);
  ok = ok && dalloc(&w.S, c * d.disc_total, false);
  ok = ok && dalloc(&w.PR, c * d.n_rows, false);
  ok = ok && dalloc(&w.gram, c * w.gram_parts * w.gram_entries, false);
  ok = ok && dalloc(&w.coef, c * nz, false);
  ok = ok && dalloc(&w.ab_fail, c, false);
  ok = ok && dalloc(&w.O, c * nn, false);
  ok = ok && dalloc(&w.T, c * (h.dark.empty() ? 1 : nn), false);
  ok = ok && dalloc(&w.PF, c * (h.dark.empty() ? 1 : nn), false);
  ok = ok && dalloc(&w.TM, c * (h.dark.empty() ? 1 : nn), false);
  ok = ok && dalloc(&w.vec_w, c * max_unknown, false);
  ok = ok && dalloc(&w.vec_x, c * max_unknown, false);
  ok = ok && dalloc(&w.vec_s, c * max_unknown, false);
  ok = ok && dalloc(&w.cg_iters, c * n_led, false);
  ok = ok && dalloc(&w.df_work, 1, false);
  if (ok) ok = cuda_ok(cudaMemset(w.df_work, 0, sizeof(unsigned long long)), "cudaMemset");
  ok = ok && dalloc(&w.TOUT, c * nn * h.u, false);
  ok = ok && dalloc(&z.bs.stats, size_t(params.max_batch) * d.n_img * 3, false);
  ok = ok && dalloc(&z.bs.live, size_t(params.max_batch), false);
  ok = ok && dalloc(&z.bs.live_count, 1, false);
  ok = ok && cuda_ok(cudaMallocHost(reinterpret_cast<void**>(&z.h_live_count), sizeof(int32_t)), "cudaMallocHost");
  if (ok) ok = cuda_ok(cudaMemset(w.cg_iters, 0, c * n_led * sizeof(int32_t)), "cudaMemset");
  if (!ok) {
    // give back what this attempt got, so that a retry (the lazily allocated second set) does not strand it
    const std::string why = g_cuda_err;                  // keep the first failure's text ("out of memory")
    for (size_t k = first_alloc; k < allocs.size(); ++k) cudaFree(allocs[k]);
    allocs.resize(first_alloc);
    workspace_bytes = bytes_before;
    if (z.h_live_count) { cudaFreeHost(z.h_live_count); z.h_live_count = nullptr; }
    z.ws = Workspace{};
    z.bs = BatchState{};
    cudaGetLastError();
    g_cuda_err = why;
  }
  z.ready = ok;
  return ok;
}

// Makes the plan's device current for the duration of a call (function attributes, allocations and launches
// are per device; a plan lives on the device that was current at apic_plan_create).
struct DeviceGuard {
  int prev = -1;
  bool ok = true;          // false: the plan's device could not be made current; the entry returns APIC_ECUDA
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) ok = cuda_ok(cudaSetDevice(dev), "cudaSetDevice(plan's device)"); else prev = -1;
    if (!ok) prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// The device-pointer entries run on workspace set 0 and share the launch counter and the profiler with the host
// pipeline: a batch that apic_submit_host left in flight is completed first (its results are then in its host
// buffers, and the caller's later apic_wait_host returns at once).
static int drain_host_slots(apic_plan* plan) {
  for (int q = 0; q < 2; ++q)
    if (plan->slot[q].busy) {
      const int rc = apic_wait_host(plan, q);
      if (rc != APIC_OK) return rc;
    }
  return APIC_OK;
}

static void fill_info(const HostTables& h, apic_plan_info_t* info) {
  std::memset(info, 0, sizeof *info);
  info->tile_n = h.n; info->upsample = h.u; info->out_n = h.n * h.u;
  info->n_bright = h.nb; info->n_dark = h.nd; info->n_zernike = h.nz;
  info->n_pairs = h.n_pairs;
  info->n_rows = int(h.row_src.size() / 2);
  info->n_grad_rows = int(h.grad_rows.size() / 2);
  info->n_union = int(h.union_f.size());
  info->n_known = h.n_known;
  info->n_dark_used = int(h.dark.size());
  for (const DarkLed& L : h.dark) {
    info->max_unknown = std::max(info->max_unknown, L.n_unknown);
    info->max_equations = std::max(info->max_equations, L.n_eq);
  }
  info->radius_bins = h.radius;
}

extern "C" {

void apic_params_default(apic_params* p) {
  std::memset(p, 0, sizeof *p);
  p->upsample = 2;
  p->kk_pad = 1;
  p->refine_iters = 3;
  p->df_iters = 48;
  p->df_tol = 1e-4f;
  p->intensity_floor = 1e-6f;
  p->bg_mode = 0;
  p->bg_threshold = 0.f;
  p->max_batch = 64;
  p->chunk_tiles = 0;
  p->df_mode = 0;
  p->df_team = 0;
  p->df_order = 0;
}

const char* apic_strerror(int err) {
  switch (err) {
    case APIC_OK: return "ok";
    case APIC_EINVAL: return g_plan_err.empty() ? "invalid parameter" : g_plan_err.c_str();
    case APIC_ECUDA: return "CUDA runtime error (see apic_last_cuda_error)";
    case APIC_ENOMEM: return "out of memory";
    case APIC_EBATCH: return "batch outside 1..max_batch";
    case APIC_ESCRATCH:
      return "more tiles than the library's built-in scratch holds (apic_reassemble_static_max_tiles); use apic_reassemble "
             "with a caller-supplied d_work";
  }
  return "unknown error";
}

const char* apic_last_cuda_error(void) { return g_cuda_err.c_str(); }
const char* apic_version(void) { return "libapic 0.1 (sm_100a)"; }

int apic_geometry_info(const apic_params* p, apic_plan_info_t* info, int* led, int* n_unknown, int* n_equations,
                       int cap) {
  if (!p || !info) return APIC_EINVAL;
  HostTables h;
  std::string err;
  if (!build_geometry(*p, h, err)) { g_plan_err = err; return APIC_EINVAL; }
  fill_info(h, info);
  for (int k = 0; k < int(h.dark.size()) && k < cap; ++k) {
    if (led) led[k] = h.dark[k].led;
    if (n_unknown) n_unknown[k] = h.dark[k].n_unknown;
    if (n_equations) n_equations[k] = h.dark[k].n_eq;
  }
  return APIC_OK;
}

int apic_geometry_dark_grids(const apic_params* p, int* mx, int* my, int cap) {
  if (!p || !mx || !my) return APIC_EINVAL;
  HostTables h;
  std::string err;
  if (!build_geometry(*p, h, err)) { g_plan_err = err; return APIC_EINVAL; }
  for (int k = 0; k < int(h.dark.size()) && k < cap; ++k) {
    mx[k] = h.dark[k].mx;
    my[k] = h.dark[k].my;
  }
  return APIC_OK;
}

int apic_plan_destroy(apic_plan* plan) {
  if (!plan) return APIC_OK;
  DeviceGuard guard(plan->pd.device);
  for (void* q : plan->allocs) cudaFree(q);
  for (cudaEvent_t e : plan->prof.ev) cudaEventDestroy(e);
  for (WsSet& z : plan->set) {
    if (z.h_live_count) cudaFreeHost(z.h_live_count);
    if (z.aux) { cudaStreamDestroy(z.aux); cudaEventDestroy(z.ev_fork); cudaEventDestroy(z.ev_join); }
  }
  cudaFree(plan->st_int); cudaFree(plan->st_field); cudaFree(plan->st_zern); cudaFree(plan->st_pupil);
  cudaFree(plan->st_status);
  cudaFree(plan->st_raw); cudaFree(plan->st_scale);
  for (auto& q : plan->slot) {
    if (q.busy) cudaEventSynchronize(q.out_done);
    cudaFree(q.in_f32); cudaFree(q.in_u16); cudaFree(q.in_scale); cudaFree(q.field); cudaFree(q.zern); cudaFree(q.pupil);
    cudaFree(q.status);
    if (q.ks) { cudaStreamDestroy(q.ks); cudaEventDestroy(q.in_done); cudaEventDestroy(q.k_done); cudaEventDestroy(q.out_done); }
  }
  if (plan->copy_in) {
    cudaStreamDestroy(plan->copy_in); cudaStreamDestroy(plan->copy_out); cudaStreamDestroy(plan->aux);
    for (cudaEvent_t e : plan->part_ev) if (e) cudaEventDestroy(e);
  }
  delete plan;
  return APIC_OK;
}

int apic_plan_create(const apic_params* p, apic_plan** out) {
  if (!p || !out) return APIC_EINVAL;
  *out = nullptr;
  int ndev = 0;
  if (!cuda_ok(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount") || ndev < 1) {
    if (g_cuda_err.empty()) g_cuda_err = "no CUDA device";
    return APIC_ECUDA;                                  // no CPU fallback
  }
  apic_plan* plan = new (std::nothrow) apic_plan;
  if (!plan) return APIC_ENOMEM;
  cudaGetDevice(&plan->pd.device);
  cudaDeviceGetAttribute(&plan->pd.sms, cudaDevAttrMultiProcessorCount, plan->pd.device);
  cudaDeviceGetAttribute(&plan->pd.l2_bytes, cudaDevAttrL2CacheSize, plan->pd.device);
  std::string err;
  if (!build_geometry(*p, plan->host, err)) {
    g_plan_err = err;
    delete plan;
    return APIC_EINVAL;
  }
  plan->params = *p;
  plan->params.k_bright = nullptr; plan->params.k_dark = nullptr; plan->params.noll = nullptr;  // copied into host tables
  const HostTables& h = plan->host;
  DevTables& d = plan->dev;
  const int n = h.n, nz = h.nz;
  d.n = n; d.u = h.u; d.nb = h.nb; d.nd = h.nd; d.nz = nz; d.n_img = h.nb + h.nd;
  bool ok = true;
  // twiddles and output ramps, fp64 -> fp32
  {
    std::vector<float2> tw;
    build_twiddles(n, tw);
    ok = ok && plan->upload(&d.tw, tw);
    d.kk_n = h.kk_n;
    d.tw_kk = d.tw;
    if (h.kk_n != n) {
      std::vector<float2> twk;
      build_twiddles(h.kk_n, twk);
      ok = ok && plan->upload(&d.tw_kk, twk);
    }
    std::vector<float2> txy, one;
    for (int r1 : {6, 8, 10, 12, 16}) {
      build_twiddles_xy(r1, one);
      txy.insert(txy.end(), one.begin(), one.end());
    }
    ok = ok && plan->upload(&d.tw_xy, txy);
    std::vector<float2> ramp(size_t(h.u) * n);
    for (int a = 0; a < h.u; ++a)
      for (int f = 0; f < n; ++f) {
        const int k = f < n / 2 ? f : f - n;
        const double ang = 2.0 * M_PI * double(k) * a / double(h.u * n);
        ramp[size_t(a) * n + f] = make_float2(float(std::cos(ang)), float(std::sin(ang)));
      }
    ok = ok && plan->upload(&d.ramp, ramp);
  }
  ok = ok && plan->upload(&d.halfplane2, h.halfplane2);
  d.disc_total = h.disc_off[h.nb];
  ok = ok && plan->upload(&d.disc_zern, h.disc_zern);
  ok = ok && plan->upload(&d.bf_col0, h.bf_col0);
  ok = ok && plan->upload(&d.bf_ncol, h.bf_ncol);
  ok = ok && plan->upload(&d.bf_map_off, h.bf_map_off);
  ok = ok && plan->upload(&d.bf_map, h.bf_map);
  d.bf_max_ncol = 0;
  for (int v : h.bf_ncol) d.bf_max_ncol = std::max(d.bf_max_ncol, v);
  d.n_rows = int(h.row_src.size() / 2);
  d.n_grad = int(h.grad_rows.size() / 2);
  ok = ok && plan->upload(&d.row_src, h.row_src);
  {
    // device copy transposed to [nz][n_rows]: consecutive threads (consecutive rows) read consecutive floats
    const size_t nr = h.a_full.size() / size_t(std::max(1, nz));
    std::vector<float> at(h.a_full.size());
    for (size_t r = 0; r < nr; ++r)
      for (int j = 0; j < nz; ++j) at[size_t(j) * nr + r] = h.a_full[r * nz + j];
    ok = ok && plan->upload(&d.a_full, at);
  }
  ok = ok && plan->upload(&d.grad_rows, h.grad_rows);
  d.n_union = int(h.union_f.size());
  ok = ok && plan->upload(&d.union_f, h.union_f);
  ok = ok && plan->upload(&d.union_off, h.union_off);
  ok = ok && plan->upload(&d.union_src, h.union_src);
  d.known_row0 = h.known_row0; d.known_nrow = h.known_nrow;
  d.n_pupil = int(h.pupil_idx.size());
  ok = ok && plan->upload(&d.pupil_idx, h.pupil_idx);
  ok = ok && plan->upload(&d.pupil_zern, h.pupil_zern);
  int max_unknown = 1;
  for (const DarkLed& L : h.dark) {
    DarkDev q{};
    q.n_unknown = L.n_unknown; q.n_disc = L.n_disc; q.n_eq = L.n_eq;
    q.d_col0 = L.d_col0; q.d_ncol = L.d_ncol; q.d_row0 = L.d_row0; q.d_nrow = L.d_nrow;
    q.u_row0 = L.u_row0; q.u_nrow = L.u_nrow;
    q.q_col0 = L.q_col0; q.q_ncol = L.q_ncol; q.q_row0 = L.q_row0; q.q_nrow = L.q_nrow;
    q.led = L.led;
    ok = ok && plan->upload(&q.disc_f, L.disc_f);
    ok = ok && plan->upload(&q.zern, L.zern);
    ok = ok && plan->upload(&q.dmap, L.dmap);
    ok = ok && plan->upload(&q.qmap, L.qmap);
    q.mx = L.mx; q.my = L.my;
    for (int st = 0; st <= kMaxUStrips; ++st)
      q.u_strip_off[st] = L.u_row_off[size_t(std::min(16 * st, L.u_nrow))];
    // (L.u_nrow + 15) / 16 <= kMaxUStrips: checked by build_geometry
    q.accumulate = L.accumulate ? 1 : 0;
    q.n_avg = int(L.avg_f.size());
    ok = ok && plan->upload(&q.avg_f, L.avg_f);
    ok = ok && plan->upload(&q.avg_w, L.avg_w);
    auto modp = [](int k, int m) { return ((k % m) + m) % m; };
    q.u0m = modp(L.u_row0, L.my); q.q0m = modp(L.q_row0, L.my); q.d0m = modp(L.d_row0, L.my);
    ok = ok && plan->upload(&q.dmap_m, L.dmap_m);
    ok = ok && plan->upload(&q.qmask_m, L.qmask_m);
    plan->dark.push_back(q);
    max_unknown = std::max(max_unknown, L.n_unknown);
  }
  ok = ok && plan->upload(&plan->d_dark, plan->dark);
  // ---- workspace: tiles per internal pass
  const size_t nn = size_t(n) * n;
  int chunk = p->chunk_tiles;
  if (chunk <= 0) {
    if (n == 256 && p->df_mode != 3 && !h.dark.empty()) {
      // reduced-grid darkfield kernel: its CG working set is ~0.3 MB per tile (TM + p_M on grids of 15-20 k bins),
      // so the pass is sized for the kernel's scheduler instead: one tile per SM, i.e. teams of two CTAs on the two
      // resident CTA slots of every SM.  Measured on config 2 (profiles/r2_darkfield.md): 148 tiles x 2 CTAs take 7.5 ms
      // per 64 tiles, 296 tiles x 1 CTA 8.5 ms
      chunk = std::max(1, plan->pd.sms);
    } else {
      // full-grid darkfield CG working set per tile: T rows in use (<= 2/3 N) + p (N^2) ~ 1.7 N^2 complex64; a pass
      // is sized to half of this device's L2
      const double per_tile = 1.7 * double(nn) * sizeof(float2);
      chunk = int(0.5 * double(std::max(plan->pd.l2_bytes, 32 << 20)) / per_tile);
      chunk = std::max(8, std::min(chunk, 512));
    }
  }
  chunk = std::max(1, std::min(chunk, p->max_batch));
  plan->chunk = chunk;
  plan->max_unknown = max_unknown;
  ok = ok && plan->alloc_set(plan->set[0]);
  if (!ok) {
    const bool oom = g_cuda_err.find("out of memory") != std::string::npos;
    apic_plan_destroy(plan);
    return oom ? APIC_ENOMEM : APIC_ECUDA;
  }
  *out = plan;
  return APIC_OK;
}

int apic_plan_info(const apic_plan* plan, apic_plan_info_t* info) {
  if (!plan || !info) return APIC_EINVAL;
  fill_info(plan->host, info);
  info->chunk_tiles = plan->chunk;
  info->table_bytes = plan->table_bytes;
  info->workspace_bytes = plan->workspace_bytes;
  return APIC_OK;
}

int apic_plan_dark_sets(const apic_plan* plan, int* led, int* n_unknown, int* n_equations) {
  if (!plan) return APIC_EINVAL;
  for (size_t k = 0; k < plan->host.dark.size(); ++k) {
    if (led) led[k] = plan->host.dark[k].led;
    if (n_unknown) n_unknown[k] = plan->host.dark[k].n_unknown;
    if (n_equations) n_equations[k] = plan->host.dark[k].n_eq;
  }
  return APIC_OK;
}

// The whole path on workspace set `zi`.  `src` holds either fp32 intensities or uint16 counts + per-image scale;
// the uint16 form is converted in the loads of S0, S1 and S8 (no fp32 working copy).
static int reconstruct_impl(apic_plan* plan, int zi, const ImgSrc& src, int batch, float* d_field, float* d_zernike,
                            float* d_pupil, int32_t* d_status, cudaStream_t s, const float* d_init = nullptr) {
  if (!plan || !(src.f32 || (src.u16 && src.scale)) || !d_field || !d_zernike || !d_status) return APIC_EINVAL;
  if (batch < 1 || batch > plan->params.max_batch) return APIC_EBATCH;
  WsSet& z = plan->set[zi];
  if (!z.ready && !plan->alloc_set(z)) return APIC_ENOMEM;
  const DevTables& t = plan->dev;
  const Workspace& w = z.ws;
  const apic_params& p = plan->params;
  if (zi == 0) plan->launches = 0;
  cudaGetLastError();
  // S0: statistics, status, list of tiles to reconstruct
  {
    LaunchCtx c{s, &plan->launches, &plan->prof, z.bs.live, z.bs.live_count, 0, batch, &plan->pd};
    launch_image_stats(t, src, batch, z.bs.stats, c);
    launch_tile_status(t, z.bs.stats, batch, p.bg_mode, p.bg_threshold, d_status, z.bs.live, z.bs.live_count, c);
    launch_zero_dead(t, d_status, batch, d_field, d_zernike, d_pupil, c);
  }
  if (d_pupil) cudaMemsetAsync(d_pupil, 0, size_t(batch) * t.n * t.n * sizeof(float2), s);
  int n_live = batch;
  if (p.bg_mode != 0) {
    cudaMemcpyAsync(z.h_live_count, z.bs.live_count, sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    if (!cuda_ok(cudaStreamSynchronize(s), "background pass")) return APIC_ECUDA;
    n_live = *z.h_live_count;
  }
  if (!z.aux) {
    if (!cuda_ok(cudaStreamCreateWithFlags(&z.aux, cudaStreamNonBlocking), "cudaStreamCreate") ||
        !cuda_ok(cudaEventCreateWithFlags(&z.ev_fork, cudaEventDisableTiming), "cudaEventCreate") ||
        !cuda_ok(cudaEventCreateWithFlags(&z.ev_join, cudaEventDisableTiming), "cudaEventCreate"))
      return APIC_ECUDA;
  }
  const int n_dark_used = int(plan->dark.size());
  // balanced passes: ceil(n_live / chunk) passes of (almost) equal size
  const int n_pass = (n_live + w.chunk - 1) / w.chunk;
  const int per_pass = n_pass ? (n_live + n_pass - 1) / n_pass : 0;
  for (int c0 = 0; c0 < n_live; c0 += per_pass) {
    LaunchCtx c{s, &plan->launches, &plan->prof, z.bs.live, z.bs.live_count, c0, std::min(per_pass, n_live - c0),
                &plan->pd, z.aux, z.ev_fork, z.ev_join};
    launch_kk(t, w, c, src, z.bs.stats, p.intensity_floor);                                   // S1-S5
    launch_aberration(t, w, c, p.refine_iters, d_zernike, d_status, d_init);                  // S6
    launch_stitch(t, w, c);                                                                   // S7
    if ((p.df_mode == 0 || p.df_mode == 5) && t.n == 256) {                                   // S8-S10
      // df_wide.cu: mode 0 = 256-thread CTAs at 128 registers (groups 11), mode 5 = 1024-thread CTA pairs (groups 4)
      if (!launch_darkfield_wide(t, plan->d_dark, plan->dark.data(), n_dark_used, w, c, src, p.df_iters, p.df_tol, p.df_team,
                                 p.df_mode == 0 ? 11 : 4))
        launch_darkfield_mgrid(t, plan->d_dark, n_dark_used, w, c, src, p.df_iters, p.df_tol, 0);
    } else if (p.df_mode == 6 && t.n == 256)
      launch_darkfield_mgrid(t, plan->d_dark, n_dark_used, w, c, src, p.df_iters, p.df_tol, p.df_team);
    else if (p.df_mode == 4 && t.n == 256)
      launch_darkfield_tma(t, plan->d_dark, plan->dark.data(), n_dark_used, w, c, src, p.df_iters, p.df_tol, p.df_team);
    else
      launch_darkfield_team(t, plan->d_dark, n_dark_used, w, c, src, p.df_iters, p.df_tol, p.df_team);
    launch_output(t, w, c, d_field, d_pupil);                                                 // S10
  }
  if (!cuda_ok(cudaGetLastError(), "apic_reconstruct launch")) return APIC_ECUDA;
  return APIC_OK;
}

int apic_reconstruct(apic_plan* plan, const float* d_intensity, int batch, float* d_field, float* d_zernike,
                     float* d_pupil, int32_t* d_status, void* cuda_stream) {
  if (!plan || !d_intensity) return APIC_EINVAL;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  if (const int rc = drain_host_slots(plan)) return rc;
  return reconstruct_impl(plan, 0, ImgSrc{d_intensity, nullptr, nullptr}, batch, d_field, d_zernike, d_pupil, d_status,
                          static_cast<cudaStream_t>(cuda_stream));
}

int apic_reconstruct_prior(apic_plan* plan, const float* d_intensity, const float* d_zernike_init, int batch, float* d_field,
                           float* d_zernike, float* d_pupil, int32_t* d_status, void* cuda_stream) {
  if (!plan || !d_intensity || !d_zernike_init) return APIC_EINVAL;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  if (const int rc = drain_host_slots(plan)) return rc;
  return reconstruct_impl(plan, 0, ImgSrc{d_intensity, nullptr, nullptr}, batch, d_field, d_zernike, d_pupil, d_status,
                          static_cast<cudaStream_t>(cuda_stream), d_zernike_init);
}

int apic_reconstruct_u16(apic_plan* plan, const uint16_t* d_raw, const float* d_scale, int batch, float* d_field,
                         float* d_zernike, float* d_pupil, int32_t* d_status, void* cuda_stream) {
  if (!plan || !d_raw || !d_scale) return APIC_EINVAL;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  if (const int rc = drain_host_slots(plan)) return rc;
  return reconstruct_impl(plan, 0, ImgSrc{nullptr, d_raw, d_scale}, batch, d_field, d_zernike, d_pupil, d_status,
                          static_cast<cudaStream_t>(cuda_stream));
}

// Host-buffer form of both entries: H2D, reconstruct, D2H, one synchronisation.
static int reconstruct_host_impl(apic_plan* plan, const float* h_intensity, const uint16_t* h_raw, const float* h_scale,
                                 int batch, float* h_field, float* h_zernike, float* h_pupil, int32_t* h_status,
                                 void* cuda_stream);

int apic_reconstruct_host(apic_plan* plan, const float* h_intensity, int batch, float* h_field, float* h_zernike,
                          float* h_pupil, int32_t* h_status, void* cuda_stream) {
  if (!h_intensity) return APIC_EINVAL;
  return reconstruct_host_impl(plan, h_intensity, nullptr, nullptr, batch, h_field, h_zernike, h_pupil, h_status, cuda_stream);
}

int apic_reconstruct_host_u16(apic_plan* plan, const uint16_t* h_raw, const float* h_scale, int batch,
                              float* h_field, float* h_zernike, float* h_pupil, int32_t* h_status, void* cuda_stream) {
  if (!h_raw || !h_scale) return APIC_EINVAL;
  return reconstruct_host_impl(plan, nullptr, h_raw, h_scale, batch, h_field, h_zernike, h_pupil, h_status, cuda_stream);
}

static bool ensure_copy_streams(apic_plan* plan);
static int reconstruct_host_impl(apic_plan* plan, const float* h_intensity, const uint16_t* h_raw, const float* h_scale,
                                 int batch, float* h_field, float* h_zernike, float* h_pupil, int32_t* h_status,
                                 void* cuda_stream) {
  if (!plan || !h_field || !h_zernike || !h_status) return APIC_EINVAL;
  if (batch < 1 || batch > plan->params.max_batch) return APIC_EBATCH;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const DevTables& t = plan->dev;
  const size_t nn = size_t(t.n) * t.n, on = size_t(t.n) * t.u;
  const size_t n_px = size_t(batch) * t.n_img * nn;
  const size_t b_field = size_t(batch) * on * on * 2 * sizeof(float);
  const size_t b_zern = size_t(batch) * t.nz * sizeof(float), b_pupil = size_t(batch) * nn * 2 * sizeof(float);
  if (batch > plan->st_batch || (h_pupil && !plan->st_has_pupil)) {
    cudaFree(plan->st_field); cudaFree(plan->st_zern); cudaFree(plan->st_pupil); cudaFree(plan->st_status);
    plan->st_field = plan->st_zern = plan->st_pupil = nullptr;
    plan->st_status = nullptr;
    plan->st_batch = 0;
    bool ok = cuda_ok(cudaMalloc(reinterpret_cast<void**>(&plan->st_field), b_field), "cudaMalloc staging") &&
              cuda_ok(cudaMalloc(reinterpret_cast<void**>(&plan->st_zern), b_zern), "cudaMalloc staging") &&
              cuda_ok(cudaMalloc(reinterpret_cast<void**>(&plan->st_status), size_t(batch) * sizeof(int32_t)), "cudaMalloc staging");
    if (ok && h_pupil) ok = cuda_ok(cudaMalloc(reinterpret_cast<void**>(&plan->st_pupil), b_pupil), "cudaMalloc staging");
    if (!ok) return APIC_ENOMEM;
    plan->st_batch = batch;
    plan->st_has_pupil = h_pupil != nullptr;
  }
  if (h_raw) {
    if (batch > plan->st_raw_batch) {
      cudaFree(plan->st_raw); cudaFree(plan->st_scale);
      plan->st_raw = nullptr; plan->st_scale = nullptr; plan->st_raw_batch = 0;
      if (!cuda_ok(cudaMalloc(reinterpret_cast<void**>(&plan->st_raw), n_px * sizeof(uint16_t)), "cudaMalloc staging") ||
          !cuda_ok(cudaMalloc(reinterpret_cast<void**>(&plan->st_scale), size_t(batch) * t.n_img * sizeof(float)), "cudaMalloc staging"))
        return APIC_ENOMEM;
      plan->st_raw_batch = batch;
    }
  } else if (batch > plan->st_int_batch) {
    cudaFree(plan->st_int);
    plan->st_int = nullptr; plan->st_int_batch = 0;
    if (!cuda_ok(cudaMalloc(reinterpret_cast<void**>(&plan->st_int), n_px * sizeof(float)), "cudaMalloc staging")) return APIC_ENOMEM;
    plan->st_int_batch = batch;
  }
  constexpr int kEv = 2 * apic_plan::kMaxParts;
  if (!ensure_copy_streams(plan)) return APIC_ECUDA;
  for (int q = 0; q < 2; ++q)                             // the synchronous entry shares the workspace sets with the slots
    if (plan->slot[q].busy && apic_wait_host(plan, q) != APIC_OK) return APIC_ECUDA;
  // Sub-batches of >= 16 tiles alternate between the plan's two workspace sets and two compute streams (the caller's
  // and one of the plan's), so that the kernels of part k run beside those of part k+1 and beside the upload of the
  // parts after it and the download of the parts before it.  Results do not depend on the split (a tile's result is
  // independent of its batch; tested).
  const int parts = std::max(1, std::min(apic_plan::kMaxParts, batch / 16));
  if (parts > 1 && !plan->alloc_set(plan->set[1])) return APIC_ENOMEM;
  const int per = (batch + parts - 1) / parts;
  const size_t img_px = size_t(t.n_img) * nn;
  cudaEventRecord(plan->part_ev[kEv], s);                                      // earlier work on the caller's stream
  cudaStreamWaitEvent(plan->copy_in, plan->part_ev[kEv], 0);
  cudaStreamWaitEvent(plan->copy_out, plan->part_ev[kEv], 0);
  cudaStreamWaitEvent(plan->aux, plan->part_ev[kEv], 0);
  for (int k = 0, b0 = 0; b0 < batch; ++k, b0 += per) {
    const int nb = std::min(per, batch - b0);
    if (h_raw) {
      cudaMemcpyAsync(plan->st_raw + b0 * img_px, h_raw + b0 * img_px, nb * img_px * sizeof(uint16_t), cudaMemcpyHostToDevice,
                      plan->copy_in);
      cudaMemcpyAsync(plan->st_scale + size_t(b0) * t.n_img, h_scale + size_t(b0) * t.n_img, size_t(nb) * t.n_img * sizeof(float),
                      cudaMemcpyHostToDevice, plan->copy_in);
    } else {
      cudaMemcpyAsync(plan->st_int + b0 * img_px, h_intensity + b0 * img_px, nb * img_px * sizeof(float), cudaMemcpyHostToDevice,
                      plan->copy_in);
    }
    cudaEventRecord(plan->part_ev[2 * k], plan->copy_in);
  }
  int rc = APIC_OK;
  for (int k = 0, b0 = 0; b0 < batch && rc == APIC_OK; ++k, b0 += per) {
    const int nb = std::min(per, batch - b0);
    const int zi = k & 1;
    cudaStream_t ks = zi ? plan->aux : s;
    cudaStreamWaitEvent(ks, plan->part_ev[2 * k], 0);
    float* f = plan->st_field + size_t(b0) * on * on * 2;
    float* z = plan->st_zern + size_t(b0) * t.nz;
    float* pu = h_pupil ? plan->st_pupil + size_t(b0) * nn * 2 : nullptr;
    int32_t* st = plan->st_status + b0;
    const ImgSrc src = h_raw ? ImgSrc{nullptr, plan->st_raw + b0 * img_px, plan->st_scale + size_t(b0) * t.n_img}
                             : ImgSrc{plan->st_int + b0 * img_px, nullptr, nullptr};
    rc = reconstruct_impl(plan, zi, src, nb, f, z, pu, st, ks);
    if (rc != APIC_OK) break;
    cudaEventRecord(plan->part_ev[2 * k + 1], ks);
    cudaStreamWaitEvent(plan->copy_out, plan->part_ev[2 * k + 1], 0);
    cudaMemcpyAsync(h_field + size_t(b0) * on * on * 2, f, size_t(nb) * on * on * 2 * sizeof(float), cudaMemcpyDeviceToHost, plan->copy_out);
    cudaMemcpyAsync(h_zernike + size_t(b0) * t.nz, z, size_t(nb) * t.nz * sizeof(float), cudaMemcpyDeviceToHost, plan->copy_out);
    if (h_pupil) cudaMemcpyAsync(h_pupil + size_t(b0) * nn * 2, pu, size_t(nb) * nn * 2 * sizeof(float), cudaMemcpyDeviceToHost, plan->copy_out);
    cudaMemcpyAsync(h_status + b0, st, size_t(nb) * sizeof(int32_t), cudaMemcpyDeviceToHost, plan->copy_out);
  }
  // the caller's stream also ends after the plan's second compute stream
  cudaEventRecord(plan->part_ev[kEv + 1], plan->aux);
  cudaStreamWaitEvent(s, plan->part_ev[kEv + 1], 0);
  bool ok = cuda_ok(cudaStreamSynchronize(plan->copy_in), "apic_reconstruct_host");
  ok = cuda_ok(cudaStreamSynchronize(plan->copy_out), "apic_reconstruct_host") && ok;
  ok = cuda_ok(cudaStreamSynchronize(plan->aux), "apic_reconstruct_host") && ok;
  ok = cuda_ok(cudaStreamSynchronize(s), "apic_reconstruct_host") && ok;
  if (rc != APIC_OK) return rc;
  return ok ? APIC_OK : APIC_ECUDA;
}

// ------------------------------------------------------------------ streaming host entries
static bool ensure_copy_streams(apic_plan* plan) {
  constexpr int kEv = 2 * apic_plan::kMaxParts;
  if (plan->copy_in) return true;
  bool ok = cuda_ok(cudaStreamCreateWithFlags(&plan->copy_in, cudaStreamNonBlocking), "cudaStreamCreate") &&
            cuda_ok(cudaStreamCreateWithFlags(&plan->copy_out, cudaStreamNonBlocking), "cudaStreamCreate") &&
            cuda_ok(cudaStreamCreateWithFlags(&plan->aux, cudaStreamNonBlocking), "cudaStreamCreate");
  for (int k = 0; ok && k < kEv + 2; ++k)
    ok = cuda_ok(cudaEventCreateWithFlags(&plan->part_ev[k], cudaEventDisableTiming), "cudaEventCreate");
  return ok;
}

static bool grow_bytes(void** p, size_t bytes) {
  cudaFree(*p);
  *p = nullptr;
  return cuda_ok(cudaMalloc(p, bytes), "cudaMalloc staging");
}
#define grow(pp, count) grow_bytes(reinterpret_cast<void**>(pp), (count) * sizeof(**(pp)))

static int submit_host_impl(apic_plan* plan, int slot, const float* h_intensity, const uint16_t* h_raw, const float* h_scale,
                            int batch, float* h_field, float* h_zernike, float* h_pupil, int32_t* h_status) {
  if (!plan || !h_field || !h_zernike || !h_status || slot < 0 || slot > 1) return APIC_EINVAL;
  if (batch < 1 || batch > plan->params.max_batch) return APIC_EBATCH;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  apic_plan::HostSlot& q = plan->slot[slot];
  if (q.busy) {                                          // a slot holds one batch at a time
    const int rc = apic_wait_host(plan, slot);
    if (rc != APIC_OK) return rc;
  }
  const DevTables& t = plan->dev;
  const size_t nn = size_t(t.n) * t.n, on = size_t(t.n) * t.u, img_px = size_t(t.n_img) * nn;
  if (!ensure_copy_streams(plan)) return APIC_ECUDA;
  if (!plan->alloc_set(plan->set[slot])) return APIC_ENOMEM;
  if (!q.ks) {
    bool ok = cuda_ok(cudaStreamCreateWithFlags(&q.ks, cudaStreamNonBlocking), "cudaStreamCreate") &&
              cuda_ok(cudaEventCreateWithFlags(&q.in_done, cudaEventDisableTiming), "cudaEventCreate") &&
              cuda_ok(cudaEventCreateWithFlags(&q.k_done, cudaEventDisableTiming), "cudaEventCreate") &&
              cuda_ok(cudaEventCreateWithFlags(&q.out_done, cudaEventDisableTiming), "cudaEventCreate");
    if (!ok) return APIC_ECUDA;
    cudaEventRecord(q.k_done, q.ks);                     // "the previous batch of this slot has read its inputs"
  }
  // staging buffers of this slot (grow-only; the slot is idle here, so nothing reads the old ones)
  if (batch > q.cap_out || (h_pupil && !q.has_pupil)) {
    bool ok = grow(&q.field, size_t(batch) * on * on * 2) && grow(&q.zern, size_t(batch) * t.nz) &&
              grow(&q.status, size_t(batch));
    if (ok && (h_pupil || q.has_pupil)) ok = grow(&q.pupil, size_t(batch) * nn * 2);
    if (!ok) { q.cap_out = 0; return APIC_ENOMEM; }
    q.cap_out = batch;
    q.has_pupil = q.has_pupil || h_pupil != nullptr;
  }
  if (h_raw && batch > q.cap_u16) {
    if (!grow(&q.in_u16, size_t(batch) * img_px) || !grow(&q.in_scale, size_t(batch) * t.n_img)) { q.cap_u16 = 0; return APIC_ENOMEM; }
    q.cap_u16 = batch;
  }
  if (!h_raw && batch > q.cap_f32) {
    if (!grow(&q.in_f32, size_t(batch) * img_px)) { q.cap_f32 = 0; return APIC_ENOMEM; }
    q.cap_f32 = batch;
  }
  // upload (one copy stream for both slots: uploads queue behind each other and beside the other slot's kernels)
  cudaStreamWaitEvent(plan->copy_in, q.k_done, 0);
  if (h_raw) {
    cudaMemcpyAsync(q.in_u16, h_raw, size_t(batch) * img_px * sizeof(uint16_t), cudaMemcpyHostToDevice, plan->copy_in);
    cudaMemcpyAsync(q.in_scale, h_scale, size_t(batch) * t.n_img * sizeof(float), cudaMemcpyHostToDevice, plan->copy_in);
  } else {
    cudaMemcpyAsync(q.in_f32, h_intensity, size_t(batch) * img_px * sizeof(float), cudaMemcpyHostToDevice, plan->copy_in);
  }
  cudaEventRecord(q.in_done, plan->copy_in);
  // kernels
  cudaStreamWaitEvent(q.ks, q.in_done, 0);
  const ImgSrc src = h_raw ? ImgSrc{nullptr, q.in_u16, q.in_scale} : ImgSrc{q.in_f32, nullptr, nullptr};
  float* pu = h_pupil ? q.pupil : nullptr;
  const int rc = reconstruct_impl(plan, slot, src, batch, q.field, q.zern, pu, q.status, q.ks);
  cudaEventRecord(q.k_done, q.ks);
  if (rc != APIC_OK) { cudaStreamSynchronize(q.ks); return rc; }
  // download
  cudaStreamWaitEvent(plan->copy_out, q.k_done, 0);
  cudaMemcpyAsync(h_field, q.field, size_t(batch) * on * on * 2 * sizeof(float), cudaMemcpyDeviceToHost, plan->copy_out);
  cudaMemcpyAsync(h_zernike, q.zern, size_t(batch) * t.nz * sizeof(float), cudaMemcpyDeviceToHost, plan->copy_out);
  if (h_pupil) cudaMemcpyAsync(h_pupil, pu, size_t(batch) * nn * 2 * sizeof(float), cudaMemcpyDeviceToHost, plan->copy_out);
  cudaMemcpyAsync(h_status, q.status, size_t(batch) * sizeof(int32_t), cudaMemcpyDeviceToHost, plan->copy_out);
  cudaEventRecord(q.out_done, plan->copy_out);
  q.busy = true;
  return cuda_ok(cudaGetLastError(), "apic_submit_host") ? APIC_OK : APIC_ECUDA;
}

int apic_submit_host(apic_plan* plan, int slot, const float* h_intensity, int batch, float* h_field, float* h_zernike,
                     float* h_pupil, int32_t* h_status) {
  if (!h_intensity) return APIC_EINVAL;
  return submit_host_impl(plan, slot, h_intensity, nullptr, nullptr, batch, h_field, h_zernike, h_pupil, h_status);
}

int apic_submit_host_u16(apic_plan* plan, int slot, const uint16_t* h_raw, const float* h_scale, int batch, float* h_field,
                         float* h_zernike, float* h_pupil, int32_t* h_status) {
  if (!h_raw || !h_scale) return APIC_EINVAL;
  return submit_host_impl(plan, slot, nullptr, h_raw, h_scale, batch, h_field, h_zernike, h_pupil, h_status);
}

int apic_wait_host(apic_plan* plan, int slot) {
  if (!plan || slot < 0 || slot > 1) return APIC_EINVAL;
  apic_plan::HostSlot& q = plan->slot[slot];
  if (!q.busy) return APIC_OK;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  q.busy = false;
  return cuda_ok(cudaEventSynchronize(q.out_done), "apic_wait_host") ? APIC_OK : APIC_ECUDA;
}

int apic_debug_buffer(const apic_plan* plan, int which, void** d_ptr, size_t* bytes_per_tile) {
  if (!plan || !d_ptr || !bytes_per_tile) return APIC_EINVAL;
  const DevTables& t = plan->dev;
  switch (which) {
    case APIC_DBG_SUBSPECTRA:
      *d_ptr = plan->set[0].ws.S; *bytes_per_tile = size_t(t.disc_total) * sizeof(float2); return APIC_OK;
    case APIC_DBG_OBJECT_SPECTRUM:
      *d_ptr = plan->set[0].ws.O; *bytes_per_tile = size_t(t.n) * t.n * sizeof(float2); return APIC_OK;
    case APIC_DBG_DF_ITERS:
      *d_ptr = plan->set[0].ws.cg_iters; *bytes_per_tile = std::max<size_t>(1, plan->dark.size()) * sizeof(int32_t); return APIC_OK;
  }
  return APIC_EINVAL;
}

int apic_debug_copy(const apic_plan* plan, int which, void* d_dst, int tiles, void* cuda_stream) {
  void* src = nullptr;
  size_t bytes = 0;
  const int rc = apic_debug_buffer(plan, which, &src, &bytes);
  if (rc != APIC_OK) return rc;
  if (!d_dst || tiles < 1 || tiles > plan->chunk) return APIC_EINVAL;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  // the stage buffers are those of workspace set 0: a batch in flight in pipeline slot 0 would be overwriting them
  if (plan->slot[0].busy && apic_wait_host(const_cast<apic_plan*>(plan), 0) != APIC_OK) return APIC_ECUDA;
  if (!cuda_ok(cudaMemcpyAsync(d_dst, src, bytes * tiles, cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(cuda_stream)),
               "apic_debug_copy"))
    return APIC_ECUDA;
  return APIC_OK;
}

// Twiddle tables of the two test entries below, one set per device (allocated on first use, never freed).
namespace {
std::mutex g_tw_mutex;
std::map<std::pair<int, int>, float2*> g_tw_cache;     // (device, table id) -> device pointer
const float2* cached_twiddles(int table, const std::vector<float2>& host) {
  int dev = 0;
  cudaGetDevice(&dev);
  std::lock_guard<std::mutex> lock(g_tw_mutex);
  auto it = g_tw_cache.find({dev, table});
  if (it != g_tw_cache.end()) return it->second;
  float2* q = nullptr;
  if (!cuda_ok(cudaMalloc(reinterpret_cast<void**>(&q), host.size() * sizeof(float2)), "cudaMalloc")) return nullptr;
  if (!cuda_ok(cudaMemcpy(q, host.data(), host.size() * sizeof(float2), cudaMemcpyHostToDevice), "cudaMemcpy")) return nullptr;
  g_tw_cache[{dev, table}] = q;
  return q;
}
}  // namespace

int apic_fft2d(float* d_data, int n, int batch, int inverse, void* cuda_stream) {
  if (!d_data || batch < 1 || !(n == 64 || n == 128 || n == 256 || n == 512)) return APIC_EINVAL;
  std::vector<float2> tw;
  build_twiddles(n, tw);
  const float2* d_tw = cached_twiddles(n, tw);
  if (!d_tw) return APIC_ECUDA;
  launch_fft2d(reinterpret_cast<float2*>(d_data), n, batch, inverse != 0, d_tw, static_cast<cudaStream_t>(cuda_stream));
  if (!cuda_ok(cudaGetLastError(), "apic_fft2d")) return APIC_ECUDA;
  return APIC_OK;
}

int apic_fft2d_xy(float* d_data, int mx, int my, int batch, int mode, void* cuda_stream) {
  auto okl = [](int l) { return l == 96 || l == 128 || l == 160 || l == 192 || l == 256; };
  if (!d_data || batch < 1 || !okl(mx) || !okl(my) || mode < 0 || mode > 3) return APIC_EINVAL;
  std::vector<float2> txy, one;
  for (int r1 : {6, 8, 10, 12, 16}) {
    build_twiddles_xy(r1, one);
    txy.insert(txy.end(), one.begin(), one.end());
  }
  const float2* tw = cached_twiddles(0, txy);
  if (!tw) return APIC_ECUDA;
  if (launch_fft2d_xy(reinterpret_cast<float2*>(d_data), mx, my, batch, mode, tw, static_cast<cudaStream_t>(cuda_stream)))
    return APIC_EINVAL;
  if (!cuda_ok(cudaGetLastError(), "apic_fft2d_xy")) return APIC_ECUDA;
  return APIC_OK;
}

int apic_last_launch_count(const apic_plan* plan) { return plan ? plan->launches : 0; }

static const char* kCatNames[CAT_COUNT] = {
    "stats_status", "kk_log_rowfft", "kk_col_mask", "kk_row_exp", "kk_col_gather", "ab_pair_products", "ab_gram",
    "ab_solve", "stitch", "out_rows", "out_cols", "pupil", "df_mgrid_kernel", "df_team_kernel", "df_tma_kernel", "df_wide_kernel"};

int apic_profile_categories(void) { return CAT_COUNT; }
const char* apic_profile_category_name(int cat) { return (cat >= 0 && cat < CAT_COUNT) ? kCatNames[cat] : ""; }

int apic_profile_begin(apic_plan* plan, int stride, int max_samples) {
  if (!plan || stride < 1 || max_samples < 1) return APIC_EINVAL;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  if (const int rc = drain_host_slots(plan)) return rc;   // the counters are per plan, not per batch in flight
  Profiler& pr = plan->prof;
  while (int(pr.ev.size()) < 2 * max_samples) {
    cudaEvent_t e;
    if (!cuda_ok(cudaEventCreate(&e), "cudaEventCreate")) return APIC_ECUDA;
    pr.ev.push_back(e);
  }
  pr.cat.assign(pr.ev.size() / 2, 0);
  pr.used = 0;
  pr.stride = stride;
  for (long long& v : pr.launches) v = 0;
  pr.on = true;
  for (WsSet& z : plan->set)
    if (z.ready && !cuda_ok(cudaMemset(z.ws.df_work, 0, sizeof(unsigned long long)), "cudaMemset")) return APIC_ECUDA;
  return APIC_OK;
}

int apic_profile_work(apic_plan* plan, unsigned long long* line_transforms) {
  if (!plan || !line_transforms) return APIC_EINVAL;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  *line_transforms = 0;
  for (WsSet& z : plan->set) {
    unsigned long long v = 0;
    if (z.ready && !cuda_ok(cudaMemcpy(&v, z.ws.df_work, sizeof v, cudaMemcpyDeviceToHost), "apic_profile_work"))
      return APIC_ECUDA;
    *line_transforms += v;
  }
  return APIC_OK;
}

int apic_profile_end(apic_plan* plan, double* ms_sum, long long* samples, long long* launches) {
  if (!plan || !ms_sum || !samples || !launches) return APIC_EINVAL;
  DeviceGuard guard(plan->pd.device);
  if (!guard.ok) return APIC_ECUDA;
  Profiler& pr = plan->prof;
  pr.on = false;
  for (int c = 0; c < CAT_COUNT; ++c) { ms_sum[c] = 0; samples[c] = 0; launches[c] = pr.launches[c]; }
  for (int i = 0; i < pr.used; ++i) {
    if (!cuda_ok(cudaEventSynchronize(pr.ev[2 * i + 1]), "cudaEventSynchronize")) return APIC_ECUDA;
    float ms = 0.f;
    if (!cuda_ok(cudaEventElapsedTime(&ms, pr.ev[2 * i], pr.ev[2 * i + 1]), "cudaEventElapsedTime")) return APIC_ECUDA;
    ms_sum[pr.cat[i]] += ms;
    samples[pr.cat[i]] += 1;
  }
  pr.used = 0;
  return APIC_OK;
}

}  // extern "C"
