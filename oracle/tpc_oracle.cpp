// ===========================================================================
// CPU ORACLE of the ALICE-HLT-style TPC sector tracker  --  TEST INFRASTRUCTURE
// ===========================================================================
// Plain, slow, single-threaded restatement of what the hot path computes:
// Cellular-Automaton seeding + Kalman fit / track following, per TPC sector
// ("Cellular Automaton principle to build track seeds: short
// track candidate of around 5 to 10 hits. Afterwards, it uses the Kalman filter
// for track fitting and track following"; L123 cluster-wise then track-wise;
// L138 sectors processed individually; L182 159 pad rows; L213 clusters are
// identified by index).  The paper prints no formula; every formula is a
// reading, written out as numbered fp32 sequences in docs/ARITH_SPEC.md
// (sections cited below as "SPEC n / tag").
//
// THIS FILE IS NOT PART OF THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may call it.  It shares
// no code, header, table or constant with paper_1712_09434_b200/csrc: the
// struct layouts and the defaults below are its own.
//
// Pins (tests/test_oracle_*.py, CPU only): exhaustive neighbour search on small
// events (neighbours_bruteforce below) == grid search; transport vs closed-form
// helix + finite-difference Jacobian; update vs matrix-form Kalman; noiseless
// helices recovered to 1e-5 (fp64 instantiation); unit pulls; mirror / batch /
// grid-size invariances; hand-built examples.
// SPEC 9 (sector-segment merger + refit) is pinned by tests/test_oracle_merge.py: rotation vs
// the closed-form helix in the neighbour's frame and vs finite differences, noiseless crossing tracks merged into
// one track with every cluster and refitted to truth (1e-5, fp64), unit pulls of the refit, no merge of
// unrelated segments, independence of the track order.
// PARITY UNPINNED: the numeric defaults (windows, cuts, initial covariance,
// gap, minimum lengths) - nothing in the paper fixes them.
//
// Build: g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC  (oracle/build.py)
// ===========================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct OGeometry {  // mirrors nothing: the oracle's own view of the detector
  int32_t n_sectors;
  int32_t n_rows;
  const float* row_x;
  float tan_half_angle;
  float z_max;
};

struct OParams {  // SPEC 8
  float sigma_y, sigma_z, nf_hy, nf_hz, nf_chi2_max, grid_bin_min, grid_bin_max, max_sinphi, c0_sinphi,
      c0_dzds, c0_qpt, accept_k2, search_max, turn_cov_scale;
  int32_t min_seed_hits, max_row_gap, min_track_hits;
  int32_t nf_z_projection;  // SPEC 1 T4/T5, SPEC 11: 0 in time-frame mode
};

enum Counter {
  CN_CLUSTERS = 0, CN_BINS, CN_NF_PAIRS, CN_START_HITS, CN_TRACKLETS_BUILT, CN_TRACKLETS_KEPT, CN_CHAIN_HITS,
  CN_SEARCH_UP, CN_SEARCH_DN, CN_CANDIDATES, CN_TRACKLET_HITS, CN_OUT_HITS, CN_OUT_TRACKS, CN_ROW_STEPS, CN_COUNT
};

template <class R> R rsqrt_(R v) { return std::sqrt(v); }
template <class R> R rabs(R v) { return std::fabs(v); }
template <class R> R rmin(R a, R b) { return std::fmin(a, b); }
template <class R> R rmax(R a, R b) { return std::fmax(a, b); }

// ---- SPEC 5: track model ---------------------------------------------------
template <class R> struct State {
  R x;
  R p[5];   // y, z, sinphi, dz/dl, q/pT
  R c[15];  // lower triangle: 00 10 11 20 21 22 30 31 32 33 40 41 42 43 44
  R chi2;
  int32_t ndf;
};

inline int tri(int i, int j) { return i >= j ? i * (i + 1) / 2 + j : j * (j + 1) / 2 + i; }

// SPEC 5.1 TRANSPORT (P1..P24). Returns false and leaves st untouched on failure.
template <class R> bool transport(State<R>& st, R xnew, R a, R max_sinphi) {
  const R y = st.p[0], z = st.p[1], s = st.p[2], t = st.p[3], q = st.p[4];
  const R dx = xnew - st.x;                                  // P1
  const R k = a * q;                                         // P2
  const R s1 = s + k * dx;                                   // P3
  if (!(rabs(s) <= max_sinphi && rabs(s1) <= max_sinphi)) return false;  // P4
  const R c = rsqrt_(R(1) - s * s);                          // P5
  const R c1 = rsqrt_(R(1) - s1 * s1);
  const R cs = c + c1;                                       // P6
  const R tt = (s + s1) / cs;                                // P7
  const R dy = dx * tt;                                      // P8
  const R dl = dx * rsqrt_(R(1) + tt * tt);                  // P9
  const R u = (R(0.5) * k) * dl;                             // P10
  const R u2 = u * u;
  const R A1 = R(0.16666667f), A2 = R(0.075f), A3 = R(0.044642857f);
  const R dS = dl * (R(1) + u2 * (A1 + u2 * (A2 + u2 * A3)));  // P11
  const R g = s * dy + c * dx;                               // P13
  const R cc = c * c1;                                       // P14
  const R f02 = g / cc;                                      // P15
  const R f04 = ((a * dx) * g) / (c1 * cs);                  // P16
  const R f12 = (t * dy) / cc;                               // P17
  const R f13 = dS;                                          // P18
  const R f14 = ((t * a) * ((R(0.5) * dx) * dy)) / cc;       // P19
  const R f24 = a * dx;                                      // P20
  const R* C = st.c;
  const R c00 = C[0], c10 = C[1], c11 = C[2], c20 = C[3], c21 = C[4], c22 = C[5], c30 = C[6], c31 = C[7],
          c32 = C[8], c33 = C[9], c40 = C[10], c41 = C[11], c42 = C[12], c43 = C[13], c44 = C[14];
  // P21 row 0 of M = F*C
  const R m00 = c00 + f02 * c20 + f04 * c40;
  const R m02 = c20 + f02 * c22 + f04 * c42;
  const R m04 = c40 + f02 * c42 + f04 * c44;
  // P22 row 1
  const R m10 = c10 + f12 * c20 + f13 * c30 + f14 * c40;
  const R m11 = c11 + f12 * c21 + f13 * c31 + f14 * c41;
  const R m12 = c21 + f12 * c22 + f13 * c32 + f14 * c42;
  const R m13 = c31 + f12 * c32 + f13 * c33 + f14 * c43;
  const R m14 = c41 + f12 * c42 + f13 * c43 + f14 * c44;
  // P23 row 2
  const R m20 = c20 + f24 * c40;
  const R m21 = c21 + f24 * c41;
  const R m22 = c22 + f24 * c42;
  const R m23 = c32 + f24 * c43;
  const R m24 = c42 + f24 * c44;
  // P24 C' = M*F^T
  R n[15];
  n[0] = m00 + f02 * m02 + f04 * m04;
  n[1] = m10 + f02 * m12 + f04 * m14;
  n[2] = m11 + f12 * m12 + f13 * m13 + f14 * m14;
  n[3] = m20 + f02 * m22 + f04 * m24;
  n[4] = m21 + f12 * m22 + f13 * m23 + f14 * m24;
  n[5] = m22 + f24 * m24;
  n[6] = c30 + f02 * c32 + f04 * c43;
  n[7] = c31 + f12 * c32 + f13 * c33 + f14 * c43;
  n[8] = c32 + f24 * c43;
  n[9] = c33;
  n[10] = c40 + f02 * c42 + f04 * c44;
  n[11] = c41 + f12 * c42 + f13 * c43 + f14 * c44;
  n[12] = c42 + f24 * c44;
  n[13] = c43;
  n[14] = c44;
  st.x = xnew;
  st.p[0] = y + dy;                                          // P12
  st.p[1] = z + dS * t;
  st.p[2] = s1;
  for (int i = 0; i < 15; ++i) st.c[i] = n[i];
  return true;
}

// SPEC 5.2 UPDATE(i, m, e) (U1..U7)
template <class R> void update(State<R>& st, int i, R m, R e) {
  const R w = R(1) / (st.c[tri(i, i)] + e);                  // U1
  const R res = m - st.p[i];                                 // U2
  R col[5], k[5];
  for (int j = 0; j < 5; ++j) col[j] = st.c[tri(j, i)];      // U3
  for (int j = 0; j < 5; ++j) k[j] = col[j] * w;             // U4
  for (int j = 0; j < 5; ++j) st.p[j] = st.p[j] + k[j] * res;  // U5
  for (int j = 0; j < 5; ++j)
    for (int l = 0; l <= j; ++l) st.c[tri(j, l)] = st.c[tri(j, l)] - k[j] * col[l];  // U6
  st.chi2 = st.chi2 + (res * res) * w;                       // U7
  st.ndf += 1;
}

// ---- tables (SPEC 1) --------------------------------------------------------
template <class R> struct Tables {
  int n_sectors, n_rows;
  std::vector<R> X, ymax, dx_up, dx_dn, ratio_up, ratio_dn;
  R a, sy2, sz2, wy, wz, smax2, z_max;
  OParams prm;
  Tables(const OGeometry& g, float bz, const OParams& p) : n_sectors(g.n_sectors), n_rows(g.n_rows), prm(p) {
    const int n = n_rows;
    X.resize(n); ymax.resize(n); dx_up.assign(n, R(0)); dx_dn.assign(n, R(0));
    ratio_up.assign(n, R(0)); ratio_dn.assign(n, R(0));
    for (int r = 0; r < n; ++r) X[r] = R(g.row_x[r]);
    for (int r = 0; r < n; ++r) ymax[r] = X[r] * R(g.tan_half_angle) + R(1);           // T1
    for (int r = 0; r + 1 < n; ++r) { dx_up[r] = X[r + 1] - X[r]; ratio_up[r] = p.nf_z_projection ? X[r + 1] / X[r] : R(1); }  // T2 T4
    for (int r = 1; r < n; ++r) { dx_dn[r] = X[r] - X[r - 1]; ratio_dn[r] = p.nf_z_projection ? X[r - 1] / X[r] : R(1); }      // T3 T5
    a = R(-0.000299792458f) * R(bz);                                                     // T6
    sy2 = R(p.sigma_y) * R(p.sigma_y); sz2 = R(p.sigma_z) * R(p.sigma_z);               // T7
    wy = R(1) / sy2; wz = R(1) / sz2;
    smax2 = R(p.search_max) * R(p.search_max);                                           // T8
    z_max = R(g.z_max);
  }
  bool a_side(int task) const { return 2 * (task % n_sectors) < n_sectors; }
};

// ---- SPEC 2: the oracle's own grid (acceleration only) ----------------------
template <class R> struct RowGrid {
  int ny = 1, nz = 1;
  R inv = 0, y0 = 0, z0 = 0;
  std::vector<uint32_t> bin_start;  // [ny*nz+1], positions into `order`
  std::vector<uint32_t> order;      // gids of the row sorted by bin
  static int clampi(R f, int n) { return (int)rmin(rmax(f, R(0)), R(n - 1)); }
  int by(R y) const { return clampi((y - y0) * inv, ny); }
  int bz(R z) const { return clampi((z - z0) * inv, nz); }
};
const float GRID_MARGIN = 0.01f;

template <class R> struct Oracle {
  const Tables<R>& T;
  const R* Y;
  const R* Z;
  const uint32_t* row_off;
  uint32_t n_clusters, n_tasks;
  std::vector<RowGrid<R>> grids;  // [n_tasks*n_rows]
  uint64_t cnt[CN_COUNT];

  Oracle(const Tables<R>& t, const R* y, const R* z, const uint32_t* ro, uint32_t n, uint32_t nt)
      : T(t), Y(y), Z(z), row_off(ro), n_clusters(n), n_tasks(nt) {
    std::memset(cnt, 0, sizeof(cnt));
    cnt[CN_CLUSTERS] = n;
  }

  // SPEC 2
  void build_grids() {
    const int nr = T.n_rows;
    grids.resize((size_t)n_tasks * nr);
    for (uint32_t task = 0; task < n_tasks; ++task)
      for (int r = 0; r < nr; ++r) {
        RowGrid<R>& G = grids[(size_t)task * nr + r];
        const uint32_t lo = row_off[(size_t)task * nr + r], hi = row_off[(size_t)task * nr + r + 1];
        const uint32_t n = hi - lo;
        const R W = R(2) * T.ymax[r], L = T.z_max + R(2);
        R B = rsqrt_((W * L) / R(n > 0 ? n : 1));
        B = rmin(rmax(B, R(T.prm.grid_bin_min)), R(T.prm.grid_bin_max));
        G.inv = R(1) / B;
        G.ny = (int)(W * G.inv) + 1;
        G.nz = (int)(L * G.inv) + 1;
        G.y0 = -T.ymax[r];
        G.z0 = T.a_side(task) ? R(-1) : -(T.z_max + R(1));
        const int nb = G.ny * G.nz;
        cnt[CN_BINS] += nb;
        G.bin_start.assign(nb + 1, 0);
        std::vector<int> b(n);
        for (uint32_t i = 0; i < n; ++i) {
          b[i] = G.bz(Z[lo + i]) * G.ny + G.by(Y[lo + i]);
          G.bin_start[b[i] + 1]++;
        }
        for (int i = 0; i < nb; ++i) G.bin_start[i + 1] += G.bin_start[i];
        G.order.resize(n);
        std::vector<uint32_t> fill(G.bin_start.begin(), G.bin_start.end() - 1);
        for (uint32_t i = 0; i < n; ++i) G.order[fill[b[i]]++] = lo + i;
      }
  }

  // visit every cluster of the grid whose bin overlaps [ylo,yhi]x[zlo,zhi]
  template <class F> void for_window(const RowGrid<R>& G, R ylo, R yhi, R zlo, R zhi, F&& f) const {
    const int iy0 = G.by(ylo), iy1 = G.by(yhi), iz0 = G.bz(zlo), iz1 = G.bz(zhi);
    for (int iz = iz0; iz <= iz1; ++iz) {
      const uint32_t b0 = G.bin_start[iz * G.ny + iy0], b1 = G.bin_start[iz * G.ny + iy1 + 1];
      for (uint32_t i = b0; i < b1; ++i) f(G.order[i]);
    }
  }

  // ---- SPEC 3: neighbour finder (N1..N5); use_grid=false is the plain definition ----
  void neighbours(int32_t* up, int32_t* dn, bool use_grid) {
    const int nr = T.n_rows;
    for (uint32_t i = 0; i < n_clusters; ++i) up[i] = dn[i] = -1;
    const R HY = R(T.prm.nf_hy), HZ = R(T.prm.nf_hz), CHI_MAX = R(T.prm.nf_chi2_max), M = R(GRID_MARGIN);
    std::vector<uint32_t> cu, cd;
    for (uint32_t task = 0; task < n_tasks; ++task)
      for (int r = 1; r + 1 < nr; ++r) {
        const size_t tr = (size_t)task * nr + r;
        const uint32_t lo = row_off[tr], hi = row_off[tr + 1];
        const uint32_t ulo = row_off[tr + 1], uhi = row_off[tr + 2], dlo = row_off[tr - 1], dhi = row_off[tr];
        const R b = T.dx_dn[r], a_ = T.dx_up[r];
        for (uint32_t h = lo; h < hi; ++h) {
          const R y = Y[h], z = Z[h];
          const R zu = z * T.ratio_up[r], zd = z * T.ratio_dn[r];                      // N1
          cu.clear(); cd.clear();
          auto test_u = [&](uint32_t u) { if (rabs(Y[u] - y) <= HY && rabs(Z[u] - zu) <= HZ) cu.push_back(u); };  // N2
          auto test_d = [&](uint32_t d) { if (rabs(Y[d] - y) <= HY && rabs(Z[d] - zd) <= HZ) cd.push_back(d); };  // N3
          if (use_grid) {
            for_window(grids[tr + 1], (y - HY) - M, (y + HY) + M, (zu - HZ) - M, (zu + HZ) + M, test_u);
            for_window(grids[tr - 1], (y - HY) - M, (y + HY) + M, (zd - HZ) - M, (zd + HZ) + M, test_d);
          } else {
            for (uint32_t u = ulo; u < uhi; ++u) test_u(u);
            for (uint32_t d = dlo; d < dhi; ++d) test_d(d);
          }
          bool have = false;
          R best = 0; uint32_t bu = 0, bd = 0;
          for (uint32_t u : cu)
            for (uint32_t d : cd) {                                                      // N4
              const R dy = ((Y[u] - y) * b) - ((y - Y[d]) * a_);
              const R dz = ((Z[u] - z) * b) - ((z - Z[d]) * a_);
              const R chi = ((dy * dy) * T.wy) + ((dz * dz) * T.wz);
              cnt[CN_NF_PAIRS]++;
              if (!(chi < CHI_MAX)) continue;                                            // N5
              if (!have || chi < best || (chi == best && (u < bu || (u == bu && d < bd)))) {
                have = true; best = chi; bu = u; bd = d;
              }
            }
          if (have) { up[h] = (int32_t)bu; dn[h] = (int32_t)bd; }
        }
      }
  }

  // ---- SPEC 4: cleaner (C1,C2) and start hits (S1) ----
  void clean(const int32_t* up, const int32_t* dn, int32_t* cu, int32_t* cd) const {
    for (uint32_t h = 0; h < n_clusters; ++h) {
      cu[h] = (up[h] >= 0 && dn[up[h]] == (int32_t)h) ? up[h] : -1;
      cd[h] = (dn[h] >= 0 && up[dn[h]] == (int32_t)h) ? dn[h] : -1;
    }
  }

  // SPEC 5.3 SEARCH (H1..H6): gid of the best cluster of (task,row) or -1
  int64_t search(const State<R>& st, uint32_t task, int row) {
    const RowGrid<R>& G = grids[(size_t)task * T.n_rows + row];
    const R y = st.p[0], z = st.p[1];
    const R ey = st.c[0] + T.sy2, ez = st.c[2] + T.sz2;                                  // H1
    const R hy2 = rmin(R(T.prm.accept_k2) * ey, T.smax2);                                // H2
    const R hz2 = rmin(R(T.prm.accept_k2) * ez, T.smax2);
    const R wy_ = rsqrt_(rmax(hy2, R(0))) + R(GRID_MARGIN), wz_ = rsqrt_(rmax(hz2, R(0))) + R(GRID_MARGIN);
    bool have = false;
    R best = 0; uint32_t bg = 0;
    for_window(G, y - wy_, y + wy_, z - wz_, z + wz_, [&](uint32_t c) {
      cnt[CN_CANDIDATES]++;
      const R dy = Y[c] - y, dz = Z[c] - z;                                              // H3
      const R dy2 = dy * dy, dz2 = dz * dz;
      if (!(dy2 <= hy2 && dz2 <= hz2)) return;                                           // H4
      const R d = (dy2 * ez) + (dz2 * ey);                                               // H5
      if (!have || d < best || (d == best && c < bg)) { have = true; best = d; bg = c; }  // H6
    });
    return have ? (int64_t)bg : -1;
  }

  void apply_hit(State<R>& st, uint32_t h) {
    update(st, 0, Y[h], T.sy2);
    update(st, 1, Z[h], T.sz2);
  }

  struct Tracklet {
    uint32_t h0;
    uint32_t task;
    int first_row, last_row, n_hits;
    State<R> st;
    std::vector<int64_t> map;  // [n_rows] gid or -1
  };

  // ---- SPEC 6: tracklet constructor (K1..K6). Returns false if chain too short (S3). ----
  bool construct(uint32_t h0, uint32_t task, int r0, const int32_t* cu, Tracklet& tk) {
    const int nr = T.n_rows;
    // S2/S3 chain length
    int len = 1;
    for (int32_t h = cu[h0]; h >= 0; h = cu[h]) ++len;
    if (len < T.prm.min_seed_hits) return false;
    cnt[CN_TRACKLETS_BUILT]++;
    cnt[CN_CHAIN_HITS] += len;
    tk.h0 = h0; tk.task = task;
    tk.map.assign(nr, -1);
    State<R>& st = tk.st;
    const uint32_t h1 = (uint32_t)cu[h0];
    {  // K1
      const R dx = T.X[r0 + 1] - T.X[r0], dy = Y[h1] - Y[h0], dz = Z[h1] - Z[h0];
      const R ri = R(1) / rsqrt_(dx * dx + dy * dy);
      st.x = T.X[r0 + 1];
      st.p[0] = Y[h1]; st.p[1] = Z[h1]; st.p[2] = dy * ri; st.p[3] = dz * ri; st.p[4] = R(0);
      for (int i = 0; i < 15; ++i) st.c[i] = R(0);
      st.c[0] = T.sy2; st.c[2] = T.sz2; st.c[5] = R(T.prm.c0_sinphi); st.c[9] = R(T.prm.c0_dzds);
      st.c[14] = R(T.prm.c0_qpt);
      st.chi2 = R(0); st.ndf = -5;
    }
    tk.map[r0] = h0; tk.map[r0 + 1] = h1;
    tk.first_row = r0; tk.last_row = r0 + 1; tk.n_hits = 2;
    bool chain_ok = true;
    {  // K2
      int r = r0 + 2;
      for (int32_t h = cu[h1]; h >= 0; h = cu[h], ++r) {
        cnt[CN_ROW_STEPS]++;
        if (!transport(st, T.X[r], T.a, R(T.prm.max_sinphi))) { chain_ok = false; break; }
        apply_hit(st, (uint32_t)h);
        tk.map[r] = h; tk.last_row = r; tk.n_hits++;
      }
    }
    if (chain_ok) {  // K3
      int gap = 0;
      for (int r = tk.last_row + 1; r < nr; ++r) {
        cnt[CN_ROW_STEPS]++;
        if (!transport(st, T.X[r], T.a, R(T.prm.max_sinphi))) break;
        cnt[CN_SEARCH_UP]++;
        const int64_t h = search(st, task, r);
        if (h >= 0) { apply_hit(st, (uint32_t)h); tk.map[r] = h; tk.last_row = r; tk.n_hits++; gap = 0; }
        else if (++gap > T.prm.max_row_gap) break;
      }
    }
    {  // K4
      if (st.x != T.X[tk.last_row]) transport(st, T.X[tk.last_row], T.a, R(T.prm.max_sinphi));
      for (int i = 0; i < 15; ++i) st.c[i] = st.c[i] * R(T.prm.turn_cov_scale);
      st.chi2 = R(0); st.ndf = -5;
      // the hit of lastRow opens the down pass, so that the final fit uses every hit of the map
      if (st.x == T.X[tk.last_row]) apply_hit(st, (uint32_t)tk.map[tk.last_row]);
    }
    {  // K5
      int gap = 0;
      for (int r = tk.last_row - 1; r >= 0; --r) {
        cnt[CN_ROW_STEPS]++;
        if (!transport(st, T.X[r], T.a, R(T.prm.max_sinphi))) break;
        if (tk.map[r] >= 0) { apply_hit(st, (uint32_t)tk.map[r]); continue; }
        cnt[CN_SEARCH_DN]++;
        const int64_t h = search(st, task, r);
        if (h >= 0) {
          apply_hit(st, (uint32_t)h); tk.map[r] = h; tk.n_hits++;
          if (r < tk.first_row) { tk.first_row = r; gap = 0; }
        } else if (r < tk.first_row) {
          if (++gap > T.prm.max_row_gap) break;
        }
      }
    }
    if (st.x != T.X[tk.first_row]) transport(st, T.X[tk.first_row], T.a, R(T.prm.max_sinphi));  // K6
    return true;
  }
};

struct OTrackOut {  // caller-allocated outputs (any pointer may be NULL)
  int32_t *link_up, *link_dn, *clean_up, *clean_dn;   // [n_clusters]
  uint32_t* start_hits;                               // [n_clusters]
  uint32_t track_capacity, hit_capacity;
  uint32_t *track_task, *track_hit_begin, *track_nhits;
  int32_t* track_ndf;
  void *track_x, *track_par, *track_cov, *track_chi2;  // R* ; par [5][cap], cov [15][cap]
  uint32_t* hit_cluster;
  // optional tracklet dump (before selection), capacity = tracklet_capacity
  uint32_t tracklet_capacity;
  uint32_t *tracklet_start, *tracklet_nhits;
  int32_t* tracklet_map;  // [cap][n_rows]
  void* tracklet_par;     // [cap][5]
  uint64_t* counters;     // [CN_COUNT]
  uint32_t n_start_hits, n_tracklets, n_tracks, n_hits;  // results
};

template <class R>
int run(const OGeometry* g, float bz, const OParams* p, uint32_t n, uint32_t nt, const R* y, const R* z,
        const uint32_t* ro, OTrackOut* o, int use_grid_nf) {
  Tables<R> T(*g, bz, *p);
  Oracle<R> O(T, y, z, ro, n, nt);
  const int nr = T.n_rows;
  O.build_grids();
  std::vector<int32_t> up(n), dn(n), cu(n), cd(n);
  O.neighbours(up.data(), dn.data(), use_grid_nf != 0);
  O.clean(up.data(), dn.data(), cu.data(), cd.data());
  // (memcpy of zero bytes from an empty vector's null data() is undefined: found by UBSan, hence the n > 0 tests)
  if (o->link_up && n) std::memcpy(o->link_up, up.data(), n * 4);
  if (o->link_dn && n) std::memcpy(o->link_dn, dn.data(), n * 4);
  if (o->clean_up && n) std::memcpy(o->clean_up, cu.data(), n * 4);
  if (o->clean_dn && n) std::memcpy(o->clean_dn, cd.data(), n * 4);
  // S1 start hits, ascending gid
  std::vector<uint32_t> starts;
  for (uint32_t h = 0; h < n; ++h)
    if (cu[h] >= 0 && cd[h] < 0) starts.push_back(h);
  O.cnt[CN_START_HITS] = starts.size();
  o->n_start_hits = (uint32_t)starts.size();
  if (o->start_hits && !starts.empty()) std::memcpy(o->start_hits, starts.data(), starts.size() * 4);
  // task,row of a gid
  std::vector<uint32_t> tr_of(n);
  for (size_t tr = 0; tr < (size_t)nt * nr; ++tr)
    for (uint32_t h = ro[tr]; h < ro[tr + 1]; ++h) tr_of[h] = (uint32_t)tr;
  // K1..K7
  std::vector<typename Oracle<R>::Tracklet> kept;
  std::vector<uint64_t> owner(n, 0), keys;
  uint32_t n_tracklets = 0;
  for (uint32_t h0 : starts) {
    typename Oracle<R>::Tracklet tk;
    const uint32_t tr = tr_of[h0];
    if (!O.construct(h0, tr / nr, (int)(tr % nr), cu.data(), tk)) continue;
    if (n_tracklets < o->tracklet_capacity) {
      const uint32_t i = n_tracklets;
      if (o->tracklet_start) o->tracklet_start[i] = h0;
      if (o->tracklet_nhits) o->tracklet_nhits[i] = tk.n_hits;
      if (o->tracklet_map) for (int r = 0; r < nr; ++r) o->tracklet_map[(size_t)i * nr + r] = (int32_t)tk.map[r];
      if (o->tracklet_par) for (int j = 0; j < 5; ++j) ((R*)o->tracklet_par)[(size_t)i * 5 + j] = tk.st.p[j];
    }
    ++n_tracklets;
    if (tk.n_hits < p->min_track_hits) continue;                                         // K6
    O.cnt[CN_TRACKLETS_KEPT]++;
    O.cnt[CN_TRACKLET_HITS] += tk.n_hits;
    const uint64_t key = ((uint64_t)tk.n_hits << 32) | (uint64_t)(0xFFFFFFFFu - h0);     // K7
    for (int r = 0; r < nr; ++r)
      if (tk.map[r] >= 0) owner[tk.map[r]] = std::max(owner[tk.map[r]], key);
    keys.push_back(key);
    kept.push_back(std::move(tk));
  }
  o->n_tracklets = n_tracklets;
  // L1..L3
  uint32_t n_tracks = 0, n_hits = 0;
  int status = 0;
  for (size_t i = 0; i < kept.size(); ++i) {
    const auto& tk = kept[i];
    std::vector<uint32_t> hits;
    for (int r = 0; r < nr; ++r)
      if (tk.map[r] >= 0 && owner[tk.map[r]] == keys[i]) hits.push_back((uint32_t)tk.map[r]);
    if ((int)hits.size() < p->min_track_hits) continue;
    if (n_tracks >= o->track_capacity || n_hits + hits.size() > o->hit_capacity) { status = 1; break; }
    const uint32_t t = n_tracks++;
    const uint32_t cap = o->track_capacity;
    if (o->track_task) o->track_task[t] = tk.task;
    if (o->track_hit_begin) o->track_hit_begin[t] = n_hits;
    if (o->track_nhits) o->track_nhits[t] = (uint32_t)hits.size();
    if (o->track_ndf) o->track_ndf[t] = tk.st.ndf;
    if (o->track_x) ((R*)o->track_x)[t] = tk.st.x;
    if (o->track_chi2) ((R*)o->track_chi2)[t] = tk.st.chi2;
    if (o->track_par) for (int j = 0; j < 5; ++j) ((R*)o->track_par)[(size_t)j * cap + t] = tk.st.p[j];
    if (o->track_cov) for (int j = 0; j < 15; ++j) ((R*)o->track_cov)[(size_t)j * cap + t] = tk.st.c[j];
    if (o->hit_cluster) for (uint32_t h : hits) o->hit_cluster[n_hits++] = h; else n_hits += hits.size();
  }
  O.cnt[CN_OUT_TRACKS] = n_tracks;
  O.cnt[CN_OUT_HITS] = n_hits;
  o->n_tracks = n_tracks;
  o->n_hits = n_hits;
  if (o->counters) std::memcpy(o->counters, O.cnt, sizeof(O.cnt));
  return status;
}

// ===========================================================================
// SPEC 9: sector-segment merger and final refit ("merges the tracks segments afterward";
// L140: the refit the paper wants on the GPU).  Written out step by step (R1..R7, G1..G7, F1..F3).
// ===========================================================================
template <class R> struct MergeTables {
  int n_half;
  R ca, sa;
  MergeTables(int n_sectors) {
    n_half = n_sectors >= 2 ? n_sectors / 2 : 1;
    const double alpha = 2.0 * 3.14159265358979323846 / (double)n_half;
    ca = (R)(float)std::cos(alpha);  // SPEC 9 tables: computed in double, rounded to fp32
    sa = (R)(float)std::sin(alpha);
    if (sizeof(R) == 8) { ca = (R)std::cos(alpha); sa = (R)std::sin(alpha); }  // fp64 instantiation: exact angle
  }
};

// SPEC 9.1 ROTATE(state, d). Returns false and leaves st untouched on failure.
template <class R> bool rotate(State<R>& st, int d, R ca, R sa_abs, R a, R max_sinphi) {
  const R sa = d > 0 ? sa_abs : -sa_abs;
  const R x = st.x, y = st.p[0], s = st.p[2], t = st.p[3], q = st.p[4];
  const R c = rsqrt_(R(1) - s * s);                            // R1
  const R s1 = s * ca - c * sa;                                // R2
  const R c1 = c * ca + s * sa;
  if (!(c1 > R(0) && rabs(s1) <= max_sinphi)) return false;    // R3
  const R j00 = ca - (s1 / c1) * sa;                           // R5
  const R j10 = -((t / c1) * sa);
  const R j20 = -((a * q) * sa);
  const R j22 = ca + (s / c) * sa;
  const R c00 = st.c[0], c10 = st.c[1], c11 = st.c[2], c20 = st.c[3], c21 = st.c[4], c22 = st.c[5], c30 = st.c[6],
          c31 = st.c[7], c32 = st.c[8], c40 = st.c[10], c41 = st.c[11], c42 = st.c[12];
  const R m00 = j00 * c00;                                     // R6
  const R m10 = j10 * c00 + c10, m11 = j10 * c10 + c11;
  const R m20 = j20 * c00 + j22 * c20, m21 = j20 * c10 + j22 * c21, m22 = j20 * c20 + j22 * c22;
  st.c[0] = m00 * j00;                                         // R7
  st.c[1] = m10 * j00; st.c[2] = m10 * j10 + m11;
  st.c[3] = m20 * j00; st.c[4] = m20 * j10 + m21; st.c[5] = m20 * j20 + m22 * j22;
  st.c[6] = c30 * j00; st.c[7] = c30 * j10 + c31; st.c[8] = c30 * j20 + c32 * j22;
  st.c[10] = c40 * j00; st.c[11] = c40 * j10 + c41; st.c[12] = c40 * j20 + c42 * j22;
  st.x = x * ca + y * sa;                                      // R4
  st.p[0] = y * ca - x * sa;
  st.p[2] = s1;
  return true;
}

struct OHit { int sector, row; uint32_t gid; };

// direction from sector `from` to its neighbour `to` (same side), SPEC 9: +1, -1, or 0 if not neighbours
inline int neighbour_dir(int from, int to, int n_half) {
  const int f = from % n_half, g = to % n_half;
  if ((from / n_half) != (to / n_half) || n_half < 2) return 0;
  if ((f + 1) % n_half == g) return +1;
  if ((g + 1) % n_half == f) return -1;
  return 0;
}

// SPEC 9.3 F1..F3 over the hits of a chain, outermost first; st = the state F1 starts from (O_im, in the frame
// of `sector`).  Returns nFit.
template <class R>
int refit_hits(const Tables<R>& T, const MergeTables<R>& MT, const std::vector<OHit>& hits, const R* Y, const R* Z,
               State<R>& st, int& sector) {
  for (int i = 0; i < 15; ++i) st.c[i] = st.c[i] * R(T.prm.turn_cov_scale);                       // F1
  st.chi2 = R(0); st.ndf = -5;
  int n_fit = 0;
  for (size_t k = 0; k < hits.size(); ++k) {                                                      // F2
    const OHit& h = hits[k];
    if (h.sector != sector) {
      const int d = neighbour_dir(sector, h.sector, MT.n_half);
      if (d == 0 || !rotate(st, d, MT.ca, MT.sa, T.a, R(T.prm.max_sinphi))) break;
      sector = h.sector;
    }
    if (st.x != T.X[h.row] && !transport(st, T.X[h.row], T.a, R(T.prm.max_sinphi))) break;
    update(st, 0, Y[h.gid], T.sy2);
    update(st, 1, Z[h.gid], T.sz2);
    ++n_fit;
  }
  return n_fit;                                                                                   // F3
}

struct OMergeIn {   // the tracks of SPEC 7 as run() wrote them
  uint32_t n_tracks, track_capacity;
  const uint32_t *track_task, *track_hit_begin, *track_nhits;
  const int32_t* track_ndf;
  const void *track_x, *track_par, *track_cov, *track_chi2;  // R*; par [5][cap], cov [15][cap]
  const uint32_t* hit_cluster;
};
struct OMergeOut {  // caller-allocated
  int32_t *next, *prev;  // [n_tracks] G6
  uint32_t merged_capacity;
  uint32_t *merged_first, *merged_nseg, *merged_nhits, *merged_nfit, *merged_sector;
  int32_t* merged_ndf;
  void *merged_x, *merged_par, *merged_cov, *merged_chi2;  // par [5][cap], cov [15][cap]
  uint32_t n_merged, n_links;
};

template <class R>
int merge_refit(const OGeometry* g, float bz, const OParams* p, float chi2_max, int32_t max_row_gap, int32_t n_slices,
                uint32_t n, uint32_t nt, const R* Y, const R* Z, const uint32_t* ro, const OMergeIn* in, OMergeOut* o) {
  Tables<R> T(*g, bz, *p);
  MergeTables<R> MT(g->n_sectors);
  const int nr = T.n_rows, ns = g->n_sectors;
  const uint32_t nT = in->n_tracks, cap = in->track_capacity;
  std::vector<uint32_t> tr_of(n);
  for (size_t tr = 0; tr < (size_t)nt * nr; ++tr)
    for (uint32_t h = ro[tr]; h < ro[tr + 1]; ++h) tr_of[h] = (uint32_t)tr;
  auto state_of = [&](uint32_t i) {
    State<R> st;
    st.x = ((const R*)in->track_x)[i];
    for (int j = 0; j < 5; ++j) st.p[j] = ((const R*)in->track_par)[(size_t)j * cap + i];
    for (int j = 0; j < 15; ++j) st.c[j] = ((const R*)in->track_cov)[(size_t)j * cap + i];
    st.chi2 = R(0); st.ndf = 0;
    return st;
  };
  std::vector<int> rf(nT), rl(nT);
  std::vector<uint32_t> gid_first(nT);
  std::vector<State<R>> outer(nT);
  std::vector<char> has_outer(nT, 0);
  for (uint32_t i = 0; i < nT; ++i) {                                                       // G1
    const uint32_t b = in->track_hit_begin[i], m = in->track_nhits[i];
    gid_first[i] = in->hit_cluster[b];
    rf[i] = (int)(tr_of[in->hit_cluster[b]] % nr);
    rl[i] = (int)(tr_of[in->hit_cluster[b + m - 1]] % nr);
    outer[i] = state_of(i);
    has_outer[i] = (outer[i].x == T.X[rl[i]] || transport(outer[i], T.X[rl[i]], T.a, R(p->max_sinphi))) ? 1 : 0;
  }
  // G2..G5: every ordered pair (plain double loop: this is the definition, not an index structure)
  std::vector<int32_t> best_out(nT, -1), best_in(nT, -1);
  std::vector<R> chi_out(nT, R(0)), chi_in(nT, R(0));
  for (uint32_t i = 0; i < nT; ++i) {
    if (!has_outer[i]) continue;
    // task = (frame*n_slices + slice)*n_sectors + sector (SPEC 11; n_slices = 1: frame = event)
    const int si = (int)(in->track_task[i] % ns), li = (int)((in->track_task[i] / ns) % n_slices),
              fi = (int)(in->track_task[i] / ns / n_slices);
    for (uint32_t j = 0; j < nT; ++j) {
      if (j == i || (int)(in->track_task[j] / ns / n_slices) != fi) continue;
      const int sj = (int)(in->track_task[j] % ns), lj = (int)((in->track_task[j] / ns) % n_slices);
      int d = 0;
      if (lj == li) {                                   // neighbouring sector of the same slice
        d = neighbour_dir(si, sj, MT.n_half);
        if (d == 0) continue;
        if (MT.n_half <= 2) d = +1;
      } else if (!(sj == si && (lj == li + 1 || lj == li - 1))) {
        continue;                                       // SPEC 11: else only the same sector of a neighbouring slice
      }
      if (!(rl[i] < rf[j] && rf[j] <= rl[i] + max_row_gap)) continue;                       // G2
      State<R> q = outer[i];                                                                // G3
      if (d != 0 && !rotate(q, d, MT.ca, MT.sa, T.a, R(p->max_sinphi))) continue;
      const State<R> sj_state = state_of(j);
      if (q.x != sj_state.x && !transport(q, sj_state.x, T.a, R(p->max_sinphi))) continue;
      R chi = R(0);                                                                         // G4
      for (int k = 0; k < 5; ++k) {
        const R dk = q.p[k] - sj_state.p[k];
        chi = chi + (dk * dk) / (q.c[tri(k, k)] + sj_state.c[tri(k, k)]);
      }
      if (!(chi < R(chi2_max))) continue;
      if (best_out[i] < 0 || chi < chi_out[i] || (chi == chi_out[i] && gid_first[j] < gid_first[best_out[i]])) {
        best_out[i] = (int32_t)j; chi_out[i] = chi;                                         // G5
      }
      if (best_in[j] < 0 || chi < chi_in[j] || (chi == chi_in[j] && gid_first[i] < gid_first[best_in[j]])) {
        best_in[j] = (int32_t)i; chi_in[j] = chi;
      }
    }
  }
  uint32_t n_links = 0;
  for (uint32_t i = 0; i < nT; ++i) { o->next[i] = -1; o->prev[i] = -1; }
  for (uint32_t i = 0; i < nT; ++i) {                                                       // G6
    const int32_t j = best_out[i];
    if (j >= 0 && best_in[j] == (int32_t)i) { o->next[i] = j; o->prev[j] = (int32_t)i; ++n_links; }
  }
  // G7 + F1..F3: chains in the order of their innermost segment
  uint32_t n_merged = 0;
  int status = 0;
  for (uint32_t i1 = 0; i1 < nT; ++i1) {
    if (o->prev[i1] >= 0) continue;
    std::vector<uint32_t> chain;
    for (int32_t k = (int32_t)i1; k >= 0; k = o->next[k]) chain.push_back((uint32_t)k);
    std::vector<OHit> hits;
    for (size_t c = chain.size(); c-- > 0;) {
      const uint32_t i = chain[c], b = in->track_hit_begin[i], m = in->track_nhits[i];
      for (uint32_t k = m; k-- > 0;) {
        const uint32_t gid = in->hit_cluster[b + k];
        hits.push_back({(int)(in->track_task[i] % ns), (int)(tr_of[gid] % nr), gid});
      }
    }
    if (n_merged >= o->merged_capacity) { status = 1; break; }
    const uint32_t im = chain.back();
    State<R> st = has_outer[im] ? outer[im] : state_of(im);
    int sector = (int)(in->track_task[im] % ns), n_fit = 0;
    if (has_outer[im]) {
      n_fit = refit_hits(T, MT, hits, Y, Z, st, sector);
    } else {  // F1: no outer end, no refit
      st.chi2 = ((const R*)in->track_chi2)[im];
      st.ndf = in->track_ndf[im];
    }
    const uint32_t mcap = o->merged_capacity, t = n_merged++;
    o->merged_first[t] = i1;
    o->merged_nseg[t] = (uint32_t)chain.size();
    o->merged_nhits[t] = (uint32_t)hits.size();
    o->merged_nfit[t] = (uint32_t)n_fit;
    o->merged_sector[t] = (uint32_t)sector;
    o->merged_ndf[t] = st.ndf;
    ((R*)o->merged_x)[t] = st.x;
    ((R*)o->merged_chi2)[t] = st.chi2;
    for (int j = 0; j < 5; ++j) ((R*)o->merged_par)[(size_t)j * mcap + t] = st.p[j];
    for (int j = 0; j < 15; ++j) ((R*)o->merged_cov)[(size_t)j * mcap + t] = st.c[j];
  }
  o->n_merged = n_merged;
  o->n_links = n_links;
  return status;
}

// ===========================================================================
// SPEC 12: ITS standalone tracker, step by step: V1..V5 tracklets, W1..W4 seed, O1..O4
// outward pass, N1..N3 inward pass.  Every search is the plain loop over all clusters of the layer (the definition).
// ===========================================================================
struct OItsGeometry { float R[6], sig_rphi[6], sig_z[6], xx0[6]; };
struct OItsParams {
  float max_sinphi_pair, max_dtan, sig_sinphi, sig_tan, sig_vtx_xy, sig_vtx_z, chi2_max, max_dx;
  float c0_sinphi, c0_dzds, c0_qpt, turn_cov_scale, max_sinphi;
  int32_t min_clusters;
};
struct OItsOut {  // caller-allocated, capacity tracks
  uint32_t capacity;
  uint32_t* event;
  int32_t* cluster;     // [cap][6] gid or -1
  uint32_t* n_clusters;
  void *frame;          // R [cap][2] ca, sa
  void *out_state, *in_state;  // R [cap][22]: x, p[5], c[15], chi2
  int32_t *out_ndf, *in_ndf;
  uint32_t n_tracklets, n_tracks;
};

template <class R>
int its_track(const OItsGeometry* g, float bz, const OItsParams* p, uint32_t n_events, const R* X, const R* Y,
              const R* Z, const uint32_t* lo, const R* vtx, OItsOut* o) {
  const R a = R(-0.000299792458f) * R(bz);                                                   // T6
  const R wphi = R(1) / (R(p->sig_sinphi) * R(p->sig_sinphi)), wtan = R(1) / (R(p->sig_tan) * R(p->sig_tan));
  R ms2[6], sr2[6], sz2[6];
  for (int l = 0; l < 6; ++l) {
    ms2[l] = (R(0.0136f) * R(0.0136f)) * R(g->xx0[l]);
    sr2[l] = R(g->sig_rphi[l]) * R(g->sig_rphi[l]);
    sz2[l] = R(g->sig_z[l]) * R(g->sig_z[l]);
  }
  const R svxy2 = R(p->sig_vtx_xy) * R(p->sig_vtx_xy), svz2 = R(p->sig_vtx_z) * R(p->sig_vtx_z);
  uint32_t n_trk = 0, n_tl = 0;
  int status = 0;
  for (uint32_t e = 0; e < n_events; ++e) {
    const R vx = vtx[3 * e], vy = vtx[3 * e + 1], vz = vtx[3 * e + 2];
    const uint32_t a0 = lo[6 * e], a1 = lo[6 * e + 1], b1 = lo[6 * e + 2];
    // ---- V1..V5
    std::vector<int64_t> best1(a1 - a0, -1), best0(b1 - a1, -1);
    std::vector<R> m1(a1 - a0, R(0)), m0(b1 - a1, R(0));
    for (uint32_t A = a0; A < a1; ++A) {
      const R ax = X[A] - vx, ay = Y[A] - vy, ra = rsqrt_(ax * ax + ay * ay), ta = (Z[A] - vz) / ra;      // V1
      for (uint32_t B = a1; B < b1; ++B) {
        const R bx = X[B] - vx, by = Y[B] - vy, rb = rsqrt_(bx * bx + by * by), tb = (Z[B] - vz) / rb;
        const R sd = (ax * by - ay * bx) / (ra * rb);                                                     // V2
        const R cd = ax * bx + ay * by;
        if (!(cd > R(0) && rabs(sd) <= R(p->max_sinphi_pair) && rabs(tb - ta) <= R(p->max_dtan))) continue;  // V3
        const R m = (sd * sd) * wphi + ((tb - ta) * (tb - ta)) * wtan;                                     // V4
        int64_t& b1A = best1[A - a0];                                                                     // V5
        if (b1A < 0 || m < m1[A - a0] || (m == m1[A - a0] && B < (uint32_t)b1A)) { b1A = B; m1[A - a0] = m; }
        int64_t& b0B = best0[B - a1];
        if (b0B < 0 || m < m0[B - a1] || (m == m0[B - a1] && A < (uint32_t)b0B)) { b0B = A; m0[B - a1] = m; }
      }
    }
    for (uint32_t A = a0; A < a1; ++A) {
      const int64_t Bq = best1[A - a0];
      if (Bq < 0 || best0[(uint32_t)Bq - a1] != (int64_t)A) continue;
      const uint32_t B = (uint32_t)Bq;
      ++n_tl;
      // ---- W1..W4
      const R ax = X[A] - vx, ay = Y[A] - vy, ra = rsqrt_(ax * ax + ay * ay);
      const R bx = X[B] - vx, by = Y[B] - vy, rb = rsqrt_(bx * bx + by * by), tb = (Z[B] - vz) / rb;
      const R ca = bx / rb, sa = by / rb;                                                                 // W1
      auto loc_x = [&](uint32_t P) { return (X[P] - vx) * ca + (Y[P] - vy) * sa; };
      auto loc_y = [&](uint32_t P) { return (Y[P] - vy) * ca - (X[P] - vx) * sa; };
      const R ox = -(vx * ca + vy * sa), oy = -(vy * ca - vx * sa);
      const R xa = loc_x(A), ya = loc_y(A), xb = rb;                                                      // W2
      const R dab = rsqrt_((xb - xa) * (xb - xa) + ya * ya);
      const R kap = -((R(2) * (ya * xb)) / ((ra * rb) * dab));
      State<R> st;                                                                                        // W3
      st.x = R(0);
      st.p[0] = R(0); st.p[1] = vz; st.p[2] = -(R(0.5) * kap) * xb; st.p[3] = tb; st.p[4] = a != R(0) ? kap / a : R(0);
      for (int i = 0; i < 15; ++i) st.c[i] = R(0);
      st.c[0] = svxy2; st.c[2] = svz2; st.c[5] = R(p->c0_sinphi); st.c[9] = R(p->c0_dzds); st.c[14] = R(p->c0_qpt);
      st.chi2 = R(0); st.ndf = -5;
      update(st, 0, R(0), svxy2);                                                                         // W4
      update(st, 1, vz, svz2);
      auto scatter = [&](int l) {
        const R th = ms2[l] * (st.p[4] * st.p[4]);
        st.c[5] = st.c[5] + th * (R(1) - st.p[2] * st.p[2]);
        st.c[9] = st.c[9] + th * ((R(1) + st.p[3] * st.p[3]) * (R(1) + st.p[3] * st.p[3]));
      };
      auto attach = [&](uint32_t P, int l) {
        if (!transport(st, loc_x(P), a, R(p->max_sinphi))) return false;
        update(st, 0, loc_y(P), sr2[l]);
        update(st, 1, Z[P], sz2[l]);
        scatter(l);
        return true;
      };
      int32_t cl[6] = {(int32_t)A, (int32_t)B, -1, -1, -1, -1};
      bool alive = attach(A, 0) && attach(B, 1);                                                          // O1
      int n_cl = 2, miss = 0;
      for (int l = 2; l < 6 && alive; ++l) {                                                              // O2
        const R Rl = R(g->R[l]);
        for (int it = 0; it < 2 && alive; ++it) {
          const R dyo = st.p[0] - oy;
          const R xt = ox + rsqrt_(rmax(Rl * Rl - dyo * dyo, R(0)));
          if (it == 1 && xt == st.x) break;
          alive = transport(st, xt, a, R(p->max_sinphi));
        }
        if (!alive) break;
        const R c = rsqrt_(R(1) - st.p[2] * st.p[2]);
        const R ey = st.c[0] + sr2[l], ez = st.c[2] + sz2[l];
        int64_t best = -1;
        R chi_best = R(0);
        for (uint32_t P = lo[6 * e + l]; P < lo[6 * e + l + 1]; ++P) {
          const R dx = loc_x(P) - st.x;
          const R dy = loc_y(P) - (st.p[0] + dx * (st.p[2] / c));
          const R dz = Z[P] - (st.p[1] + dx * (st.p[3] / c));
          const R chi = (dy * dy) / ey + (dz * dz) / ez;
          if (!(rabs(dx) <= R(p->max_dx) && chi < R(p->chi2_max))) continue;
          if (best < 0 || chi < chi_best) { best = P; chi_best = chi; }   // ascending P: ties keep the smaller gid
        }
        if (best >= 0) {
          alive = attach((uint32_t)best, l);
          cl[l] = (int32_t)best; ++n_cl; miss = 0;
        } else {
          scatter(l);
          if (++miss == 2) alive = false;
        }
      }
      if (!alive || n_cl < p->min_clusters) continue;                                                     // O3
      if (n_trk >= o->capacity) { status = 1; continue; }
      const uint32_t t = n_trk++;
      auto put = [&](void* dst, const State<R>& q) {
        R* d = (R*)dst + (size_t)t * 22;
        d[0] = q.x;
        for (int i = 0; i < 5; ++i) d[1 + i] = q.p[i];
        for (int i = 0; i < 15; ++i) d[6 + i] = q.c[i];
        d[21] = q.chi2;
      };
      o->event[t] = e; o->n_clusters[t] = (uint32_t)n_cl;
      for (int l = 0; l < 6; ++l) o->cluster[(size_t)t * 6 + l] = cl[l];
      ((R*)o->frame)[2 * t] = ca; ((R*)o->frame)[2 * t + 1] = sa;
      put(o->out_state, st); o->out_ndf[t] = st.ndf;                                                      // O4
      for (int i = 0; i < 15; ++i) st.c[i] = st.c[i] * R(p->turn_cov_scale);                              // N1
      st.chi2 = R(0); st.ndf = -5;
      for (int l = 5; l >= 0; --l) {                                                                      // N2
        if (cl[l] < 0) continue;
        const uint32_t P = (uint32_t)cl[l];
        const R xp = loc_x(P);
        if (xp != st.x && !transport(st, xp, a, R(p->max_sinphi))) break;
        update(st, 0, loc_y(P), sr2[l]);
        update(st, 1, Z[P], sz2[l]);
        scatter(l);
      }
      if (st.x != R(0)) transport(st, R(0), a, R(p->max_sinphi));                                         // N3
      put(o->in_state, st); o->in_ndf[t] = st.ndf;
    }
  }
  o->n_tracklets = n_tl;
  o->n_tracks = n_trk;
  return status;
}

}  // namespace

extern "C" {

int oracle_n_counters() { return CN_COUNT; }
size_t oracle_sizeof_out() { return sizeof(OTrackOut); }

int oracle_track_f32(const OGeometry* g, float bz, const OParams* p, uint32_t n, uint32_t nt, const float* y,
                     const float* z, const uint32_t* ro, OTrackOut* o, int use_grid_nf) {
  return run<float>(g, bz, p, n, nt, y, z, ro, o, use_grid_nf);
}
int oracle_track_f64(const OGeometry* g, float bz, const OParams* p, uint32_t n, uint32_t nt, const double* y,
                     const double* z, const uint32_t* ro, OTrackOut* o, int use_grid_nf) {
  return run<double>(g, bz, p, n, nt, y, z, ro, o, use_grid_nf);
}

// --- unit entry points for the pins -----------------------------------------
// state layout: x, p[5], c[15], chi2  (22 reals) ; ndf separately
int oracle_transport_f64(double* s22, double xnew, double a, double max_sinphi) {
  State<double> st; st.x = s22[0];
  for (int i = 0; i < 5; ++i) st.p[i] = s22[1 + i];
  for (int i = 0; i < 15; ++i) st.c[i] = s22[6 + i];
  st.chi2 = s22[21]; st.ndf = 0;
  const bool ok = transport(st, xnew, a, max_sinphi);
  s22[0] = st.x;
  for (int i = 0; i < 5; ++i) s22[1 + i] = st.p[i];
  for (int i = 0; i < 15; ++i) s22[6 + i] = st.c[i];
  return ok ? 1 : 0;
}
int oracle_transport_f32(float* s22, float xnew, float a, float max_sinphi) {
  State<float> st; st.x = s22[0];
  for (int i = 0; i < 5; ++i) st.p[i] = s22[1 + i];
  for (int i = 0; i < 15; ++i) st.c[i] = s22[6 + i];
  st.chi2 = s22[21]; st.ndf = 0;
  const bool ok = transport(st, xnew, a, max_sinphi);
  s22[0] = st.x;
  for (int i = 0; i < 5; ++i) s22[1 + i] = st.p[i];
  for (int i = 0; i < 15; ++i) s22[6 + i] = st.c[i];
  return ok ? 1 : 0;
}
void oracle_update_f64(double* s22, int32_t* ndf, int i, double m, double e) {
  State<double> st; st.x = s22[0];
  for (int j = 0; j < 5; ++j) st.p[j] = s22[1 + j];
  for (int j = 0; j < 15; ++j) st.c[j] = s22[6 + j];
  st.chi2 = s22[21]; st.ndf = *ndf;
  update(st, i, m, e);
  for (int j = 0; j < 5; ++j) s22[1 + j] = st.p[j];
  for (int j = 0; j < 15; ++j) s22[6 + j] = st.c[j];
  s22[21] = st.chi2; *ndf = st.ndf;
}
void oracle_update_f32(float* s22, int32_t* ndf, int i, float m, float e) {
  State<float> st; st.x = s22[0];
  for (int j = 0; j < 5; ++j) st.p[j] = s22[1 + j];
  for (int j = 0; j < 15; ++j) st.c[j] = s22[6 + j];
  st.chi2 = s22[21]; st.ndf = *ndf;
  update(st, i, m, e);
  for (int j = 0; j < 5; ++j) s22[1 + j] = st.p[j];
  for (int j = 0; j < 15; ++j) s22[6 + j] = st.c[j];
  s22[21] = st.chi2; *ndf = st.ndf;
}


// --- SPEC 9 -------------------------------------------------------------------
size_t oracle_sizeof_merge_in() { return sizeof(OMergeIn); }
size_t oracle_sizeof_merge_out() { return sizeof(OMergeOut); }
int oracle_merge_f32(const OGeometry* g, float bz, const OParams* p, float chi2_max, int32_t max_row_gap, int32_t n_slices,
                     uint32_t n, uint32_t nt, const float* y, const float* z, const uint32_t* ro, const OMergeIn* in,
                     OMergeOut* o) {
  return merge_refit<float>(g, bz, p, chi2_max, max_row_gap, n_slices > 0 ? n_slices : 1, n, nt, y, z, ro, in, o);
}
int oracle_merge_f64(const OGeometry* g, float bz, const OParams* p, float chi2_max, int32_t max_row_gap, int32_t n_slices,
                     uint32_t n, uint32_t nt, const double* y, const double* z, const uint32_t* ro, const OMergeIn* in,
                     OMergeOut* o) {
  return merge_refit<double>(g, bz, p, chi2_max, max_row_gap, n_slices > 0 ? n_slices : 1, n, nt, y, z, ro, in, o);
}
// ROTATE on a state laid out as x, p[5], c[15], chi2 (22 reals)
int oracle_rotate_f64(double* s22, int d, int n_sectors, double a, double max_sinphi) {
  MergeTables<double> MT(n_sectors);
  State<double> st; st.x = s22[0];
  for (int i = 0; i < 5; ++i) st.p[i] = s22[1 + i];
  for (int i = 0; i < 15; ++i) st.c[i] = s22[6 + i];
  st.chi2 = s22[21]; st.ndf = 0;
  const bool ok = rotate(st, d, MT.ca, MT.sa, a, max_sinphi);
  s22[0] = st.x;
  for (int i = 0; i < 5; ++i) s22[1 + i] = st.p[i];
  for (int i = 0; i < 15; ++i) s22[6 + i] = st.c[i];
  return ok ? 1 : 0;
}
int oracle_rotate_f32(float* s22, int d, int n_sectors, float a, float max_sinphi) {
  MergeTables<float> MT(n_sectors);
  State<float> st; st.x = s22[0];
  for (int i = 0; i < 5; ++i) st.p[i] = s22[1 + i];
  for (int i = 0; i < 15; ++i) st.c[i] = s22[6 + i];
  st.chi2 = s22[21]; st.ndf = 0;
  const bool ok = rotate(st, d, MT.ca, MT.sa, a, max_sinphi);
  s22[0] = st.x;
  for (int i = 0; i < 5; ++i) s22[1 + i] = st.p[i];
  for (int i = 0; i < 15; ++i) s22[6 + i] = st.c[i];
  return ok ? 1 : 0;
}
// SPEC 9.3 on an explicit hit list (outermost first): sector[], row[], and (y,z) per hit; s22 = the state F1
// starts from (x, p, C in the frame of sector_io), replaced by the result; returns nFit
int oracle_refit_hits_f64(const OGeometry* g, float bz, const OParams* p, uint32_t n_hits, const int32_t* sector,
                          const int32_t* row, const double* y, const double* z, double* s22, int32_t* ndf,
                          int32_t* sector_io) {
  Tables<double> T(*g, bz, *p);
  MergeTables<double> MT(g->n_sectors);
  std::vector<OHit> hits;
  for (uint32_t k = 0; k < n_hits; ++k) hits.push_back({sector[k], row[k], k});
  State<double> st; st.x = s22[0];
  for (int i = 0; i < 5; ++i) st.p[i] = s22[1 + i];
  for (int i = 0; i < 15; ++i) st.c[i] = s22[6 + i];
  int sec = *sector_io;
  const int n_fit = refit_hits(T, MT, hits, y, z, st, sec);
  s22[0] = st.x;
  for (int i = 0; i < 5; ++i) s22[1 + i] = st.p[i];
  for (int i = 0; i < 15; ++i) s22[6 + i] = st.c[i];
  s22[21] = st.chi2; *ndf = st.ndf; *sector_io = sec;
  return n_fit;
}

// --- SPEC 12 -------------------------------------------------------------------
size_t oracle_sizeof_its_out() { return sizeof(OItsOut); }
int oracle_its_f32(const OItsGeometry* g, float bz, const OItsParams* p, uint32_t n_events, const float* x, const float* y,
                   const float* z, const uint32_t* lo, const float* vtx, OItsOut* o) {
  return its_track<float>(g, bz, p, n_events, x, y, z, lo, vtx, o);
}
int oracle_its_f64(const OItsGeometry* g, float bz, const OItsParams* p, uint32_t n_events, const double* x, const double* y,
                   const double* z, const uint32_t* lo, const double* vtx, OItsOut* o) {
  return its_track<double>(g, bz, p, n_events, x, y, z, lo, vtx, o);
}
}  // extern "C"
