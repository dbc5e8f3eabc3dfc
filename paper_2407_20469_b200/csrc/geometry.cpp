// geometry.cpp - fp64 host geometry for libapic (see geometry.hpp).
//
// Citations: disc supports Eq. 7; half-plane weights Eq. 5; overlap
// sets S_il Eq. 8; rows of the difference operator Eq. 10 in a
// Noll-Zernike basis (BASELINE.json item 3); darkfield sets P, U and the linear region Q of
// Eq. 13; unknown-fraction bound.  Readings: DESIGN.md §3.
#include "geometry.hpp"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <numeric>

namespace apic {

namespace {
constexpr double kDiscRtol = 1e-9;       // R3
constexpr double kHalfplaneTau = 1e-4;   // R5
constexpr double kOrderQuantum = 1e-6;   // R15
constexpr double kMaxUnknown = 0.42;

double factorial(int n) {
  double f = 1.0;
  for (int i = 2; i <= n; ++i) f *= i;
  return f;
}

struct Mask {
  int n;
  std::vector<uint8_t> v;
  explicit Mask(int n_) : n(n_), v(size_t(n_) * n_, 0) {}
  uint8_t& at(int iy, int ix) { return v[size_t(iy) * n + ix]; }
  uint8_t at(int iy, int ix) const { return v[size_t(iy) * n + ix]; }
  int count() const { return int(std::count(v.begin(), v.end(), uint8_t(1))); }
};

struct Run { int y, x0, x1; };  // centred indices, inclusive

std::vector<Run> runs_of(const Mask& m) {
  std::vector<Run> r;
  for (int y = 0; y < m.n; ++y) {
    int x = 0;
    while (x < m.n) {
      if (!m.at(y, x)) { ++x; continue; }
      int x0 = x;
      while (x < m.n && m.at(y, x)) ++x;
      r.push_back({y, x0, x - 1});
    }
  }
  return r;
}

// {a - b : a in A, b in B} on the centred grid; false if a difference would leave (-N/2, N/2).
bool minkowski_difference(const Mask& a, const Mask& b, Mask& out) {
  const int n = a.n, w = 2 * n + 2;
  std::vector<int32_t> diff(size_t(2 * n) * w, 0);
  const std::vector<Run> rb = runs_of(b);
  for (int ay = 0; ay < n; ++ay)
    for (int ax = 0; ax < n; ++ax) {
      if (!a.at(ay, ax)) continue;
      for (const Run& r : rb) {
        int dy = ay - r.y + n;               // in [1, 2n-1]
        int lo = ax - r.x1 + n, hi = ax - r.x0 + n;
        diff[size_t(dy) * w + lo] += 1;
        diff[size_t(dy) * w + hi + 1] -= 1;
      }
    }
  std::fill(out.v.begin(), out.v.end(), 0);
  bool ok = true;
  for (int dy = 0; dy < 2 * n; ++dy) {
    int acc = 0;
    for (int dx = 0; dx < 2 * n + 1; ++dx) {
      acc += diff[size_t(dy) * w + dx];
      if (acc > 0) {
        int ry = dy - n, rx = dx - n;        // the difference vector
        if (std::abs(ry) >= n / 2 || std::abs(rx) >= n / 2) { ok = false; continue; }
        out.at(ry + n / 2, rx + n / 2) = 1;
      }
    }
  }
  return ok;
}

inline int fft_index(int n, int kx, int ky) { return ((ky + n) % n) * n + ((kx + n) % n); }

}  // namespace

void noll_to_nm(int j, int& n, int& m) {
  n = 0;
  int j1 = j - 1;
  while (j1 > n) { ++n; j1 -= n; }
  int am = (n % 2 == 0) ? 2 * ((j1 + 1) / 2) : 2 * (j1 / 2) + 1;
  m = (am == 0) ? 0 : ((j % 2 == 0) ? am : -am);
}

double zernike_noll(int j, double x, double y) {
  int n, m;
  noll_to_nm(j, n, m);
  const int am = std::abs(m);
  const double rho = std::hypot(x, y), th = std::atan2(y, x);
  double rad = 0.0;
  for (int s = 0; s <= (n - am) / 2; ++s) {
    double c = ((s & 1) ? -1.0 : 1.0) * factorial(n - s) /
               (factorial(s) * factorial((n + am) / 2 - s) * factorial((n - am) / 2 - s));
    rad += c * std::pow(rho, n - 2 * s);
  }
  if (m == 0) return std::sqrt(n + 1.0) * rad;
  const double ang = (m > 0) ? std::cos(am * th) : std::sin(am * th);
  return std::sqrt(2.0 * (n + 1.0)) * rad * ang;
}

bool build_geometry(const apic_params& p, HostTables& t, std::string& err) {
  char buf[256];
  const int n = p.tile_n;
  if (!(n == 64 || n == 128 || n == 256 || n == 512)) { err = "tile_n must be 64, 128, 256 or 512"; return false; }
  if (p.upsample < 1 || p.upsample > 4) { err = "upsample must be 1..4"; return false; }
  if (!(p.wavelength_um > 0) || !(p.pixel_um > 0) || !(p.na_obj > 0)) { err = "optics must be positive"; return false; }
  if (p.n_bright < 3 || !p.k_bright) { err = "need >= 3 NA-matching LEDs"; return false; }
  if (p.n_dark < 0 || (p.n_dark > 0 && !p.k_dark)) { err = "k_dark missing"; return false; }
  if (p.n_zernike < 1 || p.n_zernike > 64 || !p.noll) { err = "n_zernike must be 1..64"; return false; }
  if (p.kk_pad != 1 && p.kk_pad != 2) { err = "kk_pad must be 1 or 2"; return false; }
  if (p.kk_pad * p.tile_n > 512) { err = "kk_pad 2 needs tile_n <= 256 (line transforms exist up to 512 points)"; return false; }
  if (p.refine_iters < 0 || p.refine_iters > 16) { err = "refine_iters must be 0..16"; return false; }
  if (p.df_iters < 1) { err = "df_iters must be >= 1"; return false; }
  if (p.bg_mode < 0 || p.bg_mode > 2) { err = "bg_mode must be 0, 1 or 2"; return false; }
  if (p.max_batch < 1) { err = "max_batch must be >= 1"; return false; }
  if (p.df_mode != 0 && (p.df_mode < 3 || p.df_mode > 6)) { err = "df_mode must be 0 (default: reduced cyclic grids at N = 256), 3 (full N x N grid), 4 (async-proxy staging), 5 (1024-thread CTA pairs, decimated CG loop) or 6 (round-1 reduced-grid kernel)"; return false; }
  if (p.df_order != 0 && p.df_order != 1) { err = "df_order must be 0 (sequential, R15) or 1 (ring-wise, R15b)"; return false; }
  if (!(p.df_team == 0 || p.df_team == 1 || p.df_team == 2 || p.df_team == 4 || p.df_team == 8)) {
    err = "df_team must be 0 (auto), 1, 2, 4 or 8"; return false;
  }
  for (int a = 0; a < p.n_zernike; ++a) {
    if (p.noll[a] < 4) { err = "Noll indices must be >= 4 (piston/tilt are the null space of Eq. 10)"; return false; }
    for (int b = 0; b < a; ++b)
      if (p.noll[a] == p.noll[b]) { err = "repeated Noll index"; return false; }
  }

  t = HostTables();
  t.n = n; t.u = p.upsample; t.nb = p.n_bright; t.nd = p.n_dark; t.nz = p.n_zernike;
  t.noll.assign(p.noll, p.noll + p.n_zernike);
  const double scale = double(n) * p.pixel_um;                 // kappa = k * N * dx
  t.radius = p.na_obj * n * p.pixel_um / p.wavelength_um;      // R = NA N dx / lambda
  const double R = t.radius, R2 = R * R * (1.0 + kDiscRtol);
  const int h = n / 2, nz = t.nz;
  t.kappa_b.resize(size_t(2) * t.nb);
  t.kappa_d.resize(size_t(2) * t.nd);
  double reach = 0;
  for (int i = 0; i < t.nb; ++i) {
    t.kappa_b[2 * i] = p.k_bright[2 * i] * scale;
    t.kappa_b[2 * i + 1] = p.k_bright[2 * i + 1] * scale;
    double kk = std::hypot(t.kappa_b[2 * i], t.kappa_b[2 * i + 1]);
    if (std::fabs(kk - R) > 0.5) {
      snprintf(buf, sizeof buf, "NA-matching LED %d: |kappa|=%.3f bins but R=%.3f (NA-matching condition, PAPER.md:82)", i, kk, R);
      err = buf; return false;
    }
    reach = std::max(reach, kk);
  }
  for (int i = 0; i < t.nd; ++i) {
    t.kappa_d[2 * i] = p.k_dark[2 * i] * scale;
    t.kappa_d[2 * i + 1] = p.k_dark[2 * i + 1] * scale;
    double kk = std::hypot(t.kappa_d[2 * i], t.kappa_d[2 * i + 1]);
    if (!(kk > R)) { snprintf(buf, sizeof buf, "darkfield LED %d is not darkfield (|kappa| <= R)", i); err = buf; return false; }
    reach = std::max(reach, kk);
  }
  if (reach + R >= h - 1) {
    snprintf(buf, sizeof buf, "synthetic aperture (%.1f bins) does not fit the raw grid (N/2 = %d)", reach + R, h);
    err = buf; return false;
  }

  auto disc_mask = [&](const double* kap, Mask& m) {
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        double dx = (ix - h) + kap[0], dy = (iy - h) + kap[1];
        m.at(iy, ix) = (dx * dx + dy * dy <= R2) ? 1 : 0;
      }
  };
  auto zern_at = [&](int j, int kx, int ky, const double* kap) {
    return zernike_noll(j, (kx + kap[0]) / R, (ky + kap[1]) / R);
  };

  // ------------------------------------------------------------------ NA-matching discs
  std::vector<Mask> discs;
  std::vector<std::vector<int32_t>> entry_of(t.nb);   // centred linear index -> flattened entry or -1
  t.disc_off.assign(t.nb + 1, 0);
  t.bf_col0.resize(t.nb); t.bf_ncol.resize(t.nb);
  t.bf_map_off.assign(t.nb + 1, 0);
  const int M = p.kk_pad * n, hm = M / 2;              // grid of the KK step (R7): bins of the N grid are a subset of it
  t.kk_n = M;
  t.halfplane2.assign(size_t(t.nb) * M * M, 0);
  for (int i = 0; i < t.nb; ++i) {
    const double* kap = &t.kappa_b[2 * i];
    Mask m(n);
    disc_mask(kap, m);
    if (!m.at(h, h)) { snprintf(buf, sizeof buf, "NA-matching LED %d: DC bin outside its disc", i); err = buf; return false; }
    entry_of[i].assign(size_t(n) * n, -1);
    int c0 = n, c1 = -1;
    const double theta0[2] = {0, 0};
    (void)theta0;
    std::vector<double> zk(nz);
    for (int a = 0; a < nz; ++a) zk[a] = zern_at(t.noll[a], 0, 0, kap);   // Z_j(kappa_i): theta_i terms
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        if (!m.at(iy, ix)) continue;
        int kx = ix - h, ky = iy - h;
        entry_of[i][size_t(iy) * n + ix] = int32_t(t.disc_f.size());
        t.disc_f.push_back(fft_index(n, kx, ky));
        for (int a = 0; a < nz; ++a) t.disc_zern.push_back(float(zern_at(t.noll[a], kx, ky, kap) - zk[a]));
        c0 = std::min(c0, kx); c1 = std::max(c1, kx);
      }
    t.disc_off[i + 1] = int32_t(t.disc_f.size());
    t.bf_col0[i] = c0; t.bf_ncol[i] = c1 - c0 + 1;
    t.bf_map_off[i + 1] = t.bf_map_off[i] + M * t.bf_ncol[i];
    t.bf_map.resize(t.bf_map_off[i + 1], -1);
    for (int iy = 0; iy < n; ++iy)
      for (int c = 0; c < t.bf_ncol[i]; ++c) {
        int kx = c0 + c, ky = iy - h, fy = (ky + M) % M;
        t.bf_map[size_t(t.bf_map_off[i]) + size_t(fy) * t.bf_ncol[i] + c] = entry_of[i][size_t(iy) * n + (kx + h)];
      }
    // Eq. 5 weights on the KK grid, FFT order
    const double kn = std::hypot(kap[0], kap[1]);
    uint8_t* w2 = &t.halfplane2[size_t(i) * M * M];
    for (int ky = -hm; ky < hm; ++ky)
      for (int kx = -hm; kx < hm; ++kx) {
        uint8_t v;
        if (kx == -hm || ky == -hm) v = 1;
        else {
          double d = (kx * kap[0] + ky * kap[1]) / kn;
          v = (d < -kHalfplaneTau) ? 2 : ((d > kHalfplaneTau) ? 0 : 1);
        }
        w2[fft_index(M, kx, ky)] = v;
      }
    discs.push_back(std::move(m));
  }

  // ------------------------------------------------------------------ pairs, rows (Eq. 8-10)
  for (int i = 0; i < t.nb; ++i)
    for (int l = i + 1; l < t.nb; ++l) {
      int cnt = 0;
      for (size_t q = 0; q < size_t(n) * n; ++q) cnt += (discs[i].v[q] & discs[l].v[q]);
      if (cnt < 2) continue;
      ++t.n_pairs;
      const double* ki = &t.kappa_b[2 * i];
      const double* kl = &t.kappa_b[2 * l];
      std::vector<int32_t> row_of(size_t(n) * n, -1);
      std::vector<double> z0(nz);
      for (int a = 0; a < nz; ++a) z0[a] = -zern_at(t.noll[a], 0, 0, ki) + zern_at(t.noll[a], 0, 0, kl);
      const int first = int(t.row_src.size() / 2);
      for (int iy = 0; iy < n; ++iy)
        for (int ix = 0; ix < n; ++ix) {
          size_t q = size_t(iy) * n + ix;
          if (!(discs[i].v[q] & discs[l].v[q])) continue;
          row_of[q] = int32_t(t.row_src.size() / 2);
          t.row_src.push_back(entry_of[i][q]);
          t.row_src.push_back(entry_of[l][q]);
          int kx = ix - h, ky = iy - h;
          for (int a = 0; a < nz; ++a)
            t.a_full.push_back(float(zern_at(t.noll[a], kx, ky, ki) - zern_at(t.noll[a], kx, ky, kl) + z0[a]));
        }
      (void)first;
      for (int axis = 0; axis < 2; ++axis)
        for (int iy = 0; iy < n; ++iy)
          for (int ix = 0; ix < n; ++ix) {
            size_t q = size_t(iy) * n + ix;
            if (row_of[q] < 0) continue;
            int y2 = iy + (axis == 1), x2 = ix + (axis == 0);
            if (y2 >= n || x2 >= n) continue;
            int32_t r1 = row_of[size_t(y2) * n + x2];
            if (r1 < 0) continue;
            t.grad_rows.push_back(row_of[q]);
            t.grad_rows.push_back(r1);
          }
    }
  if (t.n_pairs < 1) { err = "no overlapping NA-matching pair (Eq. 8)"; return false; }

  // ------------------------------------------------------------------ union + cover lists
  Mask known(n);
  t.union_off.push_back(0);
  for (int iy = 0; iy < n; ++iy)
    for (int ix = 0; ix < n; ++ix) {
      size_t q = size_t(iy) * n + ix;
      bool any = false;
      for (int i = 0; i < t.nb; ++i)
        if (discs[i].v[q]) { t.union_src.push_back(entry_of[i][q]); any = true; }
      if (any) {
        known.at(iy, ix) = 1;
        t.union_f.push_back(fft_index(n, ix - h, iy - h));
        t.union_off.push_back(int32_t(t.union_src.size()));
      }
    }

  // ------------------------------------------------------------------ darkfield sets (R15, R16)
  std::vector<std::pair<long long, int>> order;
  for (int i = 0; i < t.nd; ++i)
    order.push_back({llround(std::hypot(t.kappa_d[2 * i], t.kappa_d[2 * i + 1]) / kOrderQuantum), i});
  std::stable_sort(order.begin(), order.end());
  // df_order 1 (R15b): the LEDs of a ring (equal |kappa| key) all see the known set as it stands when the ring starts
  const bool ring_wise = p.df_order == 1;
  Mask base = known;                       // known set the current ring's LEDs are solved against
  std::vector<int> cover(size_t(n) * n, 0);
  int ring = -1;
  long long ring_key = 0;
  size_t ring_first = 0;                   // index in t.dark of the ring's first LED
  auto close_ring = [&]() {
    if (!ring_wise || t.dark.size() == ring_first) return;
    DarkLed& last = t.dark.back();
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        const int c = cover[size_t(iy) * n + ix];
        if (c >= 2) { last.avg_f.push_back(fft_index(n, ix - h, iy - h)); last.avg_w.push_back(1.0f / float(c)); }
      }
    std::fill(cover.begin(), cover.end(), 0);
  };
  for (auto& oi : order) {
    const int led = oi.second;
    if (ring < 0 || oi.first != ring_key) {
      close_ring();
      ++ring; ring_key = oi.first; ring_first = t.dark.size();
      base = known;
    }
    const Mask& ref = ring_wise ? base : known;
    const double* kap = &t.kappa_d[2 * led];
    Mask d(n), P(n), U(n);
    disc_mask(kap, d);
    int nU = 0, nD = 0;
    for (size_t q = 0; q < size_t(n) * n; ++q) {
      if (!d.v[q]) continue;
      ++nD;
      if (ref.v[q]) P.v[q] = 1; else { U.v[q] = 1; ++nU; }
    }
    if (nU == 0) continue;
    DarkLed L;
    L.led = led; L.kappa[0] = kap[0]; L.kappa[1] = kap[1];
    L.ring = ring; L.accumulate = ring_wise;
    L.unknown_fraction = double(nU) / nD;
    if (L.unknown_fraction > kMaxUnknown) {
      snprintf(buf, sizeof buf, "darkfield LED %d: unknown fraction %.3f > 0.42 (PAPER.md:201)", led, L.unknown_fraction);
      err = buf; return false;
    }
    Mask cross(n), other(n), self(n), Q(n);
    bool ok = minkowski_difference(U, P, cross);    // supp(U * P) = {u - p}
    ok = minkowski_difference(P, U, other) && ok;   // supp(P * U) = {p - u}
    ok = minkowski_difference(U, U, self) && ok;    // supp(U * U) = {u - u'}
    if (!ok) { snprintf(buf, sizeof buf, "darkfield LED %d: index-set difference wraps around the grid", led); err = buf; return false; }
    int nQ = 0;
    for (size_t q = 0; q < size_t(n) * n; ++q) {
      Q.v[q] = (cross.v[q] && !other.v[q] && !self.v[q]) ? 1 : 0;
      nQ += Q.v[q];
    }
    if (nQ == 0) { snprintf(buf, sizeof buf, "darkfield LED %d: empty linear region Q (Eq. 13)", led); err = buf; return false; }
    L.n_unknown = nU; L.n_disc = nD; L.n_eq = nQ;
    // bboxes
    auto bbox = [&](const Mask& m, int& c0, int& nc, int& r0, int& nr) {
      int x0 = n, x1 = -1, y0 = n, y1 = -1;
      for (int iy = 0; iy < n; ++iy)
        for (int ix = 0; ix < n; ++ix)
          if (m.at(iy, ix)) { x0 = std::min(x0, ix); x1 = std::max(x1, ix); y0 = std::min(y0, iy); y1 = std::max(y1, iy); }
      c0 = x0 - h; nc = x1 - x0 + 1; r0 = y0 - h; nr = y1 - y0 + 1;
    };
    bbox(d, L.d_col0, L.d_ncol, L.d_row0, L.d_nrow);
    bbox(U, L.u_col0, L.u_ncol, L.u_row0, L.u_nrow);
    if ((L.u_nrow + 15) / 16 > kMaxUStrips) {
      snprintf(buf, sizeof buf, "darkfield LED %d: its unknown set spans %d rows, more than the %d the darkfield kernels' strip "
               "table holds (pupil radius too large for this tile_n)", led, L.u_nrow, 16 * kMaxUStrips);
      err = buf; return false;
    }
    bbox(Q, L.q_col0, L.q_ncol, L.q_row0, L.q_nrow);
    // disc entries: U first (row-major), then P (row-major)
    std::vector<int32_t> ent(size_t(n) * n, -1);
    L.disc_f.resize(nD);
    L.zern.resize(size_t(nD) * nz);
    int eu = 0, ep = nU;
    L.u_row_off.assign(size_t(L.u_nrow) + 1, 0);
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        size_t q = size_t(iy) * n + ix;
        if (!d.v[q]) continue;
        if (U.v[q]) ++L.u_row_off[size_t(iy - h - L.u_row0) + 1];
        int e = U.v[q] ? eu++ : ep++;
        ent[q] = e;
        int kx = ix - h, ky = iy - h;
        L.disc_f[e] = fft_index(n, kx, ky);
        for (int a = 0; a < nz; ++a) L.zern[size_t(e) * nz + a] = float(zern_at(t.noll[a], kx, ky, kap));
      }
    for (int r = 0; r < L.u_nrow; ++r) L.u_row_off[size_t(r) + 1] += L.u_row_off[size_t(r)];
    L.dmap.assign(size_t(n) * L.d_ncol, -1);
    for (int iy = 0; iy < n; ++iy)
      for (int c = 0; c < L.d_ncol; ++c) {
        int fy = ((iy - h) + n) % n;
        L.dmap[size_t(fy) * L.d_ncol + c] = ent[size_t(iy) * n + (L.d_col0 + c + h)];
      }
    L.qmap.assign(size_t(n) * L.q_ncol, -1);
    int mq = 0;
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix) {
        if (!Q.at(iy, ix)) continue;
        int fy = ((iy - h) + n) % n;
        L.qmap[size_t(fy) * L.q_ncol + (ix - h - L.q_col0)] = mq++;
      }
    {
      // reduced cyclic grid: per axis the lags u - p - k (u in U, p in P, k in Q) must stay inside (-m, m)
      int pc0, pnc, pr0, pnr;
      bbox(P, pc0, pnc, pr0, pnr);
      auto extent = [](int u0, int un, int p0, int pn, int q0, int qn) {
        const int hi = (u0 + un - 1) - p0 - q0, lo = u0 - (p0 + pn - 1) - (q0 + qn - 1);
        return std::max(std::abs(hi), std::abs(lo));
      };
      const int ex = extent(L.u_col0, L.u_ncol, pc0, pnc, L.q_col0, L.q_ncol);
      const int ey = extent(L.u_row0, L.u_nrow, pr0, pnr, L.q_row0, L.q_nrow);
      auto pick = [&](int e) {
        const int cand[5] = {3 * n / 8, n / 2, 5 * n / 8, 3 * n / 4, n};
        for (int c : cand)
          if (c > e && c >= L.d_ncol && c >= L.d_nrow) return c;
        return n;
      };
      L.mx = pick(ex); L.my = pick(ey);
      L.dmap_m.assign(size_t(L.mx) * L.my, -1);
      L.qmask_m.assign(size_t(L.mx) * L.my, 0);
      auto pos = [&](int kx, int ky) {
        return size_t(((ky % L.my) + L.my) % L.my) * L.mx + size_t(((kx % L.mx) + L.mx) % L.mx);
      };
      for (int iy = 0; iy < n; ++iy)
        for (int ix = 0; ix < n; ++ix) {
          const size_t q = size_t(iy) * n + ix;
          if (d.v[q]) L.dmap_m[pos(ix - h, iy - h)] = ent[q];
          if (Q.v[q]) L.qmask_m[pos(ix - h, iy - h)] = 1;
        }
    }
    for (size_t q = 0; q < size_t(n) * n; ++q) { known.v[q] |= U.v[q]; cover[q] += U.v[q]; }
    t.dark.push_back(std::move(L));
  }
  close_ring();
  t.n_known = known.count();
  {
    int x0 = n, x1 = -1, y0 = n, y1 = -1;
    for (int iy = 0; iy < n; ++iy)
      for (int ix = 0; ix < n; ++ix)
        if (known.at(iy, ix)) { x0 = std::min(x0, ix); x1 = std::max(x1, ix); y0 = std::min(y0, iy); y1 = std::max(y1, iy); }
    t.known_col0 = x0 - h; t.known_ncol = x1 - x0 + 1;
    t.known_row0 = y0 - h; t.known_nrow = y1 - y0 + 1;
  }

  // ------------------------------------------------------------------ pupil output table
  const double zero[2] = {0, 0};
  for (int iy = 0; iy < n; ++iy)
    for (int ix = 0; ix < n; ++ix) {
      int kx = ix - h, ky = iy - h;
      if (double(kx) * kx + double(ky) * ky > R2) continue;
      t.pupil_idx.push_back(iy * n + ix);
      for (int a = 0; a < nz; ++a) t.pupil_zern.push_back(float(zern_at(t.noll[a], kx, ky, zero)));
    }
  return true;
}

}  // namespace apic
