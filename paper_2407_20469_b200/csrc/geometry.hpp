// geometry.hpp - host-side (fp64) geometry of the APIC path: everything that depends only on
// (N, R, kappa_i) and is therefore identical for every tile ("vectorised
// construction" taken to its end: index sets become plan-time constants).
//
// Index conventions: a "centred" index (iy, ix) is bin (kx, ky) = (ix - N/2, iy - N/2); an "FFT
// order" linear index is ((ky mod N) * N + (kx mod N)).  Compact orders of every set are the
// row-major order of the centred grid.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/apic.h"

namespace apic {

// The darkfield kernels walk the rows of an LED's unknown set U in strips of 16; their per-LED strip table has this many
// entries.  A disc spans <= 2R + 1 <= 0.34 N rows: <= 11 strips at N = 512.  build_geometry rejects what does not fit.
constexpr int kMaxUStrips = 16;

struct DarkLed {
  int led = 0;                 // input index
  double kappa[2] = {0, 0};
  int n_unknown = 0;           // |U|: disc entries [0, n_unknown) are U, the rest are P
  int n_disc = 0;              // |D_i| = |U| + |P|
  int n_eq = 0;                // |Q|
  int d_col0 = 0, d_ncol = 0;  // centred kx range of the disc bbox
  int d_row0 = 0, d_nrow = 0;  // centred ky range
  int u_col0 = 0, u_ncol = 0;  // bbox of U only
  int u_row0 = 0, u_nrow = 0;
  int q_col0 = 0, q_ncol = 0;  // bbox of Q
  int q_row0 = 0, q_nrow = 0;
  std::vector<int32_t> disc_f; // [n_disc] FFT-order linear index of each disc entry
  std::vector<int32_t> u_row_off; // [u_nrow+1] first U entry of each row of the U bbox (U entries are row-major)
  // ring-wise order (apic_params.df_order 1, reading R15b): the LED ADDS its solution to the object spectrum; the last
  // LED of a ring carries the bins of the ring solved by c >= 2 LEDs, which are then scaled by 1 / c
  int ring = 0;
  bool accumulate = false;
  std::vector<int32_t> avg_f;  // FFT-order linear index
  std::vector<float> avg_w;    // 1 / c
  std::vector<float> zern;     // [n_disc][nz] Z_j(K + kappa)
  std::vector<int32_t> dmap;   // [N (fy)][d_ncol] -> disc entry or -1
  std::vector<int32_t> qmap;   // [N (fy)][q_ncol] -> equation index or -1
  double unknown_fraction = 0;
  // Reduced cyclic grid (df_mgrid.cu): the mat-vecs of Eq. 13 only need correlations at lags in Q, so a
  // cyclic grid of mx x my bins is alias-free as soon as mx, my exceed the extent of U - P - Q per axis.
  // mx, my in {3N/8, N/2, 5N/8, 3N/4, N}; bin (kx, ky) sits at ((ky mod my) * mx + (kx mod mx)).
  int mx = 0, my = 0;
  std::vector<int32_t> dmap_m; // [my][mx] -> disc entry or -1
  std::vector<uint8_t> qmask_m;// [my][mx] -> 1 on Q
};

struct HostTables {
  int n = 0, u = 1, nb = 0, nd = 0, nz = 0;
  int kk_n = 0;                             // grid of the KK step: kk_pad * N (R7); halfplane2 and bf_map live on it
  double radius = 0;
  std::vector<double> kappa_b, kappa_d;     // [nb][2], [nd][2] in bins
  std::vector<int> noll;

  // ---- NA-matching side
  std::vector<uint8_t> halfplane2;          // [nb][kk_n*kk_n] FFT order, 2*w of Eq. 5 in {0,1,2}
  std::vector<int32_t> disc_off;            // [nb+1] offsets into the flattened sub-spectrum vector
  std::vector<int32_t> disc_f;              // [disc_off[nb]] FFT-order index of each entry
  std::vector<float> disc_zern;             // [disc_off[nb]][nz]  Z_j(K+kappa_i) - Z_j(kappa_i)
  std::vector<int32_t> bf_col0, bf_ncol;    // [nb] centred kx range of each disc
  std::vector<int32_t> bf_map_off;          // [nb+1] offsets into bf_map
  std::vector<int32_t> bf_map;              // per LED [kk_n (fy)][ncol] -> flattened entry or -1

  // ---- aberration system (Eq. 8-10)
  int n_pairs = 0;
  std::vector<int32_t> row_src;             // [rows][2] flattened sub-spectrum entries (i side, l side)
  std::vector<float> a_full;                // [rows][nz]
  std::vector<int32_t> grad_rows;           // [grows][2] (r0, r1): row r1 is the +x or +y neighbour of r0

  // ---- stitching
  std::vector<int32_t> union_f;             // [n_union] FFT-order index
  std::vector<int32_t> union_off;           // [n_union+1]
  std::vector<int32_t> union_src;           // flattened sub-spectrum entries covering each bin

  // ---- darkfield, in processing order
  std::vector<DarkLed> dark;
  int n_known = 0;
  int known_col0 = 0, known_ncol = 0;       // centred kx bbox of the final known region
  int known_row0 = 0, known_nrow = 0;       // centred ky bbox

  // ---- pupil output
  std::vector<int32_t> pupil_idx;           // centred linear index of bins with |k| <= R
  std::vector<float> pupil_zern;            // [n][nz] Z_j(k)
};

// Returns true on success; on failure `err` explains (-> APIC_EINVAL).
bool build_geometry(const apic_params& p, HostTables& t, std::string& err);

// Noll-normalised Zernike polynomial Z_j at pupil coordinate (x, y) (unit disc), fp64.
double zernike_noll(int j, double x, double y);
void noll_to_nm(int j, int& n, int& m);

}  // namespace apic
